// pack.cu -- canonical <-> device layout conversion (hot path row a1 of SURVEY.md section 8).
//
// Spinor: canonical [site][s][spin][colour][reim]  <->  device pair[s][row][k/2][h][k&1]: row = x1 +
//         L1*(x2 + L2*x3) is a lattice line along x0, h = x0>>1 the site of the parity on that line,
//         so the cb site x>>1 is row*Lh + h; a site has 12 slots k of two reals; slots 2j, 2j+1 of
//         a site are adjacent (one 128-bit vector in fp32).  One such block per parity; a FULL
//         field is the even block followed by the odd block (canonical site x -> parity p(x)).
//         fp64: complex[s][row][k][h], k = spin*3 + colour: one plane per component, a site's complex
//         number (re, im) is one 128-bit vector.
//         fp32: slot k = 4*colour + t holds one real part of a PAIR OF SPINS: t = 0: (re psi_0c,
//         re psi_1c), 1: (im psi_0c, im psi_1c), 2: (re psi_2c, re psi_3c), 3: (im psi_2c,
//         im psi_3c).  The packed f32x2 arithmetic of dhop_staged.cu then multiplies a link
//         element (a scalar) into both spin components of a half spinor at once and never needs a
//         half-negated operand (dhop_staged.cu, "arithmetic").
// Gauge : canonical [x][mu][a][b][reim]  ->  for each output parity p and each output site of that
//         parity (cb index x>>1) the 8 links that site multiplies with:
//            leg 2*mu   : U_mu(x)                       (forward hop,  psi(x+mu))
//            leg 2*mu+1 : U_mu(x-mu)^dagger             (backward hop, psi(x-mu))
//         each times -1 when the hop wraps around an antiperiodic time direction (times 0 with an open time
//         boundary, DWF_OPEN_T: the slab operator of halo.cu), stored planar
//         row by row as complex[row][f/2][h][f&1], f = leg*9 + a*3+b (the 72 link components of
//         the Lh output sites of a row are one contiguous 576*Lh-byte block, in 128-bit pairs).
//         Every canonical link appears exactly once in each parity set, so one half-Dhop reads
//         the whole gauge field once.
#include "dwf_internal.cuh"

namespace dwf {

// FULL = true: canonical sites are lexicographic x, the device field is [parity][s][row][k/2][h][k&1]
// FULL = false: canonical sites are the cb sites of one parity, the device field is [s][row][k/2][h][k&1]
template <typename T, bool IMPORT, bool FULL>
__global__ void __launch_bounds__(256)
spinor_reorder_kernel(const T *__restrict__ src, T *__restrict__ dst, const Lattice lat, const long long row0, const long long nrow_c)
{
    // one thread per complex element of the DEVICE layout (coalesced on the device side).  The call covers
    // the lattice lines row0 .. row0 + nrow_c - 1; the canonical pointer (src on import, dst on export) is
    // RELATIVE to the first site of that range (chunked host transfers, api.cu)
    using V = typename std::conditional<sizeof(T) == 4, float2, double2>::type;
    const long long Vh = lat.Vh;
    const long long nrow = Vh / lat.Lh;
    const long long n = (FULL ? 2 : 1) * nrow_c * lat.Lh * lat.Ls * 12;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n;
         e += (long long)gridDim.x * blockDim.x) {
        // fp32 device element e = ((((par*Ls + s)*nrow + row)*6 + k/2)*Lh + h)*2 + (k&1)
        // fp64 device element e =  (((par*Ls + s)*nrow + row)*12 + k)*Lh + h
        long long r = e;
        int h, k;
        if constexpr (sizeof(T) == 4) {
            const int klo = (int)(r & 1); r >>= 1;
            h = (int)(r % lat.Lh); r /= lat.Lh;
            k = 2 * (int)(r % 6) + klo; r /= 6;
        } else {
            h = (int)(r % lat.Lh); r /= lat.Lh;
            k = (int)(r % 12); r /= 12;
        }
        const long long rowc = r % nrow_c; r /= nrow_c;
        const long long row = row0 + rowc;
        const int s = (int)(r % lat.Ls);
        const int par = (int)(r / lat.Ls);
        const long long cb = rowc * lat.Lh + h;          // canonical site, relative to the chunk
        long long site = cb;
        if (FULL) {
            // lexicographic x of cb site `cb` of parity `par`: x0 = 2*h + ((x1+x2+x3+par)&1)
            long long q = row;
            const int x1 = (int)(q % lat.L[1]); q /= lat.L[1];
            const int x2 = (int)(q % lat.L[2]);
            const int x3 = (int)(q / lat.L[2]);
            site = 2 * cb + ((x1 + x2 + x3 + par) & 1);
        }
        if constexpr (sizeof(T) == 8) {
            const long long c = ((site * lat.Ls + s) * 12 + k);     // canonical complex index
            const long long d = ((((long long)par * lat.Ls + s) * nrow + row) * 12 + k) * lat.Lh + h;   // device complex index
            if (IMPORT) reinterpret_cast<V *>(dst)[d] = reinterpret_cast<const V *>(src)[c];
            else        reinterpret_cast<V *>(dst)[c] = reinterpret_cast<const V *>(src)[d];
        } else {
            // fp32: slot k = 4*colour + t holds the spin pair (2*(t/2), 2*(t/2)+1) of one real part:
            // t = 0 (re of spins 0,1), 1 (im of 0,1), 2 (re of 2,3), 3 (im of 2,3)
            const int col = k >> 2, t = k & 3;
            const long long i0 = (((site * lat.Ls + s) * 12 + ((t >> 1) * 6 + col)) << 1) + (t & 1);   // canonical real
            const long long d = (((((long long)par * lat.Ls + s) * nrow + row) * 6 + (k >> 1)) * lat.Lh + h) * 2 + (k & 1);
            if (IMPORT) reinterpret_cast<V *>(dst)[d] = V{src[i0], src[i0 + 6]};
            else {
                const V v = reinterpret_cast<const V *>(src)[d];
                dst[i0] = v.x;
                dst[i0 + 6] = v.y;
            }
        }
    }
}

// fp32: one thread per device site (parity, s, row, h): the 24 reals of a site are one 96-byte record
// on the canonical side (six 128-bit accesses per thread, whole sectors) and six 128-bit vectors on
// the device side (consecutive threads = consecutive h: coalesced).
template <bool IMPORT, bool FULL>
__global__ void __launch_bounds__(256)
spinor_reorder_sites_kernel(const float *__restrict__ src, float *__restrict__ dst, const Lattice lat, const long long row0,
                            const long long nrow_c)
{
    const long long Vh = lat.Vh;
    const long long nrow = Vh / lat.Lh;
    const long long n = (FULL ? 2 : 1) * nrow_c * lat.Lh * lat.Ls;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n;
         e += (long long)gridDim.x * blockDim.x) {
        long long r = e;
        const int h = (int)(r % lat.Lh); r /= lat.Lh;
        const long long rowc = r % nrow_c; r /= nrow_c;
        const long long row = row0 + rowc;
        const int s = (int)(r % lat.Ls);
        const int par = (int)(r / lat.Ls);
        const long long cb = rowc * lat.Lh + h;          // canonical site, relative to the chunk
        long long site = cb;
        if (FULL) {
            long long q = row;
            const int x1 = (int)(q % lat.L[1]); q /= lat.L[1];
            const int x2 = (int)(q % lat.L[2]);
            const int x3 = (int)(q / lat.L[2]);
            site = 2 * cb + ((x1 + x2 + x3 + par) & 1);
        }
        const long long canon = (site * lat.Ls + s) * 6;                                   // in float4
        const long long dev = (((long long)par * lat.Ls + s) * nrow + row) * 6 * lat.Lh + h;   // in float4: + j * Lh
        float c[24];
        if (IMPORT) {
#pragma unroll
            for (int j = 0; j < 6; j++) {
                const float4 q = reinterpret_cast<const float4 *>(src)[canon + j];
                c[4 * j] = q.x; c[4 * j + 1] = q.y; c[4 * j + 2] = q.z; c[4 * j + 3] = q.w;
            }
#pragma unroll
            for (int j = 0; j < 6; j++) {       // vector j = slots 2j, 2j+1; slot k = 4*col + t
                float v[4];
#pragma unroll
                for (int u = 0; u < 2; u++) {
                    const int k = 2 * j + u, col = k >> 2, t = k & 3;
                    const int i0 = ((t >> 1) * 6 + col) * 2 + (t & 1);
                    v[2 * u] = c[i0];
                    v[2 * u + 1] = c[i0 + 6];
                }
                reinterpret_cast<float4 *>(dst)[dev + (long long)j * lat.Lh] = make_float4(v[0], v[1], v[2], v[3]);
            }
        } else {
#pragma unroll
            for (int j = 0; j < 6; j++) {
                const float4 q = reinterpret_cast<const float4 *>(src)[dev + (long long)j * lat.Lh];
                const float v[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
                for (int u = 0; u < 2; u++) {
                    const int k = 2 * j + u, col = k >> 2, t = k & 3;
                    const int i0 = ((t >> 1) * 6 + col) * 2 + (t & 1);
                    c[i0] = v[2 * u];
                    c[i0 + 6] = v[2 * u + 1];
                }
            }
#pragma unroll
            for (int j = 0; j < 6; j++)
                reinterpret_cast<float4 *>(dst)[canon + j] = make_float4(c[4 * j], c[4 * j + 1], c[4 * j + 2], c[4 * j + 3]);
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(256)
gauge_pack_kernel(const T *__restrict__ U, T *__restrict__ set_even, T *__restrict__ set_odd,
                  const Lattice lat, const int bc_time)
{
    // one thread per (lexicographic site x, leg)
    const long long n = lat.V4 * 8;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n;
         e += (long long)gridDim.x * blockDim.x) {
        const long long x = e % lat.V4;
        const int leg = (int)(e / lat.V4);
        const int mu = leg >> 1;
        const bool bwd = leg & 1;
        int c[4];
        long long r = x;
        c[0] = (int)(r % lat.L[0]); r /= lat.L[0];
        c[1] = (int)(r % lat.L[1]); r /= lat.L[1];
        c[2] = (int)(r % lat.L[2]); r /= lat.L[2];
        c[3] = (int)r;
        const int par = (c[0] + c[1] + c[2] + c[3]) & 1;
        T *set = par ? set_odd : set_even;
        const long long cb = x >> 1;

        T sign = 1;
        long long src_site = x;
        if (bwd) {
            int cm[4] = {c[0], c[1], c[2], c[3]};
            cm[mu] = (c[mu] == 0) ? lat.L[mu] - 1 : c[mu] - 1;
            src_site = cm[0] + (long long)lat.L[0] * (cm[1] + (long long)lat.L[1] * (cm[2] + (long long)lat.L[2] * cm[3]));
            if (bc_time && mu == 3 && c[3] == 0) sign = bc_time == DWF_OPEN_T ? 0 : -1;
        } else {
            if (bc_time && mu == 3 && c[3] == lat.L[3] - 1) sign = bc_time == DWF_OPEN_T ? 0 : -1;
        }
        const T *u = U + (src_site * 4 + mu) * 18;
        const long long row = cb / lat.Lh;
        const int h = (int)(cb % lat.Lh);
        T *rowbase = set + (size_t)row * 72 * 2 * lat.Lh;
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) {
                T re, im;
                if (bwd) { re = u[(b * 3 + a) * 2]; im = -u[(b * 3 + a) * 2 + 1]; }   // dagger
                else     { re = u[(a * 3 + b) * 2]; im =  u[(a * 3 + b) * 2 + 1]; }
                const int f = leg * 9 + a * 3 + b;   // link component 0..71, stored in pairs
                const size_t off = (((size_t)(f >> 1) * lat.Lh + h) * 2 + (f & 1)) * 2;
                rowbase[off] = sign * re;
                rowbase[off + 1] = sign * im;
            }
    }
}

static int grid_for(long long n, int sm_count)
{
    long long b = (n + 255) / 256;
    long long cap = (long long)sm_count * 16;
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

// 12-real link storage: rows 0 and 1 of each of the 8 links of a site, taken from the packed
// 18-real set: complex[row][f'/2][h][f'&1], f' = leg*6 + a*3 + b (a < 2).  The staged kernel rebuilds row 2 =
// conj(row0 x row1) (times the folded boundary sign) when it loads the links of a tile.
__global__ void __launch_bounds__(256)
gauge_compress12_kernel(const float2 *__restrict__ full, float2 *__restrict__ c12, const long long nrow, const int Lh)
{
    const long long n = nrow * Lh * 48;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        // destination element e = ((row*24 + f'/2)*Lh + h)*2 + (f'&1)
        long long r = e;
        const int lo = (int)(r & 1); r >>= 1;
        const int h = (int)(r % Lh); r /= Lh;
        const int fp = 2 * (int)(r % 24) + lo;
        const long long row = r / 24;
        const int leg = fp / 6, ab = fp % 6;
        const int f = leg * 9 + ab;
        c12[e] = full[((row * 36 + (f >> 1)) * Lh + h) * 2 + (f & 1)];
    }
}

int launch_compress_gauge12(const dwf_geometry *g, cudaStream_t st)
{
    const long long nrow = g->lat.Vh / g->lat.Lh;
    for (int p = 0; p < 2; p++) {
        gauge_compress12_kernel<<<grid_for(nrow * g->lat.Lh * 48, g->sm_count), 256, 0, st>>>(
            static_cast<const float2 *>(g->gauge[p]), static_cast<float2 *>(g->gauge12[p]), nrow, g->lat.Lh);
        count_launch();
    }
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

int launch_pack_gauge(const dwf_geometry *g, const void *U_dev, cudaStream_t st)
{
    const int grid = grid_for(g->lat.V4 * 8, g->sm_count);
    if (g->prec == DWF_F32)
        gauge_pack_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float *>(U_dev), static_cast<float *>(g->gauge[0]),
                                                      static_cast<float *>(g->gauge[1]), g->lat, g->bc_time);
    else
        gauge_pack_kernel<double><<<grid, 256, 0, st>>>(static_cast<const double *>(U_dev), static_cast<double *>(g->gauge[0]),
                                                       static_cast<double *>(g->gauge[1]), g->lat, g->bc_time);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

template <bool IMPORT>
static int launch_reorder(const dwf_geometry *g, const void *src, void *dst, int parity, cudaStream_t st, long long row0,
                          long long nrow_c)
{
    const bool full = parity == DWF_FULL;
    if (nrow_c < 0) { row0 = 0; nrow_c = g->lat.Vh / g->lat.Lh; }
    const long long nsite = (full ? 2 : 1) * nrow_c * g->lat.Lh * g->lat.Ls;
    const int grid = grid_for(nsite * 12, g->sm_count);
    if (g->prec == DWF_F32) {
        auto *a = static_cast<const float *>(src);
        auto *b = static_cast<float *>(dst);
        const int gs = grid_for(nsite, g->sm_count);
        if (full) spinor_reorder_sites_kernel<IMPORT, true><<<gs, 256, 0, st>>>(a, b, g->lat, row0, nrow_c);
        else      spinor_reorder_sites_kernel<IMPORT, false><<<gs, 256, 0, st>>>(a, b, g->lat, row0, nrow_c);
    } else {
        auto *a = static_cast<const double *>(src);
        auto *b = static_cast<double *>(dst);
        if (full) spinor_reorder_kernel<double, IMPORT, true><<<grid, 256, 0, st>>>(a, b, g->lat, row0, nrow_c);
        else      spinor_reorder_kernel<double, IMPORT, false><<<grid, 256, 0, st>>>(a, b, g->lat, row0, nrow_c);
    }
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

// row0, nrow_c: the lattice lines covered (nrow_c < 0: all); the canonical pointer is relative to the first site of the range
int launch_import(const dwf_geometry *g, const void *canonical_dev, int parity, void *field, cudaStream_t st, long long row0,
                  long long nrow_c)
{
    return launch_reorder<true>(g, canonical_dev, field, parity, st, row0, nrow_c);
}
int launch_export(const dwf_geometry *g, const void *field, int parity, void *canonical_dev, cudaStream_t st, long long row0,
                  long long nrow_c)
{
    return launch_reorder<false>(g, field, canonical_dev, parity, st, row0, nrow_c);
}

// out = a x + b out over nreal reals (128-bit vectors; nreal is a multiple of 24).  The unfused path of
// dwf_dhop_oe_axpy / dwf_dhop_eo_axpy (fp64, shapes without a staged variant); x may be out.
template <typename T>
__global__ void __launch_bounds__(256)
axpby_kernel(const T *__restrict__ x, T *__restrict__ out, const T a, const T b, const size_t nvec)
{
    using V = typename std::conditional<sizeof(T) == 4, float4, double2>::type;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        const V p = reinterpret_cast<const V *>(x)[i];
        V q = reinterpret_cast<V *>(out)[i];
        q.x = fma(b, q.x, a * p.x);
        q.y = fma(b, q.y, a * p.y);
        if constexpr (sizeof(T) == 4) {
            q.z = fma(b, q.z, a * p.z);
            q.w = fma(b, q.w, a * p.w);
        }
        reinterpret_cast<V *>(out)[i] = q;
    }
}

int launch_axpby(const dwf_geometry *g, const void *x, void *out, double a, double b, size_t nreal, cudaStream_t st)
{
    const int nb = g->sm_count * 8;
    if (g->prec == DWF_F32)
        axpby_kernel<float><<<nb, 256, 0, st>>>(static_cast<const float *>(x), static_cast<float *>(out), (float)a, (float)b, nreal / 4);
    else
        axpby_kernel<double><<<nb, 256, 0, st>>>(static_cast<const double *>(x), static_cast<double *>(out), a, b, nreal / 2);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

}  // namespace dwf

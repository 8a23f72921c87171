// dwf5d.cu -- the rest of the red-black Shamir domain-wall operator ("all kernels involved
// in the DWF Dirac operator", section 4, L250 Fig.5, L254 Fig.6 -- named there, never
// printed; the definition is DESIGN.md reading #22):
//
//   (M psi)(x,s) = (5 - M5) psi(x,s) - 1/2 (Dhop psi)(x,s) - P_- psi(x,s+1) - P_+ psi(x,s-1)
//   P_+- = (1 +- gamma5)/2,   psi(x,Ls) = -m psi(x,0),   psi(x,-1) = -m psi(x,Ls-1)
//
// Mooee = everything but Dhop: diagonal in the 4D site and in colour, a bidiagonal (plus one corner)
// real matrix in s for each chirality.  gamma5 = diag(+,+,-,-), so spins 0,1 see psi(s-1) and spins
// 2,3 see psi(s+1) -- and in both device layouts a 128-bit vector holds one chirality only (fp32:
// vector j of a site is spins 0,1 for even j, spins 2,3 for odd j; fp64: component k = spin*3 + colour).
// With s the SLOWEST index of a field the fifth-dimension operators are pure streaming passes: one
// thread owns one 128-bit vector of a slice, loads it from all Ls slices (Ls independent coalesced
// loads), does the s-recurrence in registers and stores Ls vectors: one read and one write of the
// field, the minimum.  Reversing the direction of the walk (s -> Ls-1-s) turns the P_- stencil into
// the P_+ one, so both chiralities (and the adjoint, which swaps them) run the same code without
// divergence.
//   Mooee        y(0) = d x(0) + m x(Ls-1),  y(i) = d x(i) - x(i-1)                      d = 5 - M5
//   Mooee^{-1}   T = sum_{j>=1} k^{Ls-j} x(j) (Horner),  y(0) = k (x(0) - m T) / (1 + m k^Ls),
//                y(i) = k (x(i) + y(i-1))                                               k = 1/d
// (the cyclic bidiagonal system solved exactly: a forward substitution whose start value follows from
// closing the cycle).  On top: the full matrix M on full fields, the Schur complement
// S = Mooee - 1/4 D_pq Mooee^{-1} D_qp on one parity (four kernels: Dhop, Mooee^{-1}, Mooee, and
// a x + b Dhop fused in the staged kernel's epilogue), and conjugate gradients on S^dag S.
#include <math.h>
#include <type_traits>

#include "dwf_internal.cuh"
#include "reduce.cuh"

namespace dwf {

template <typename T> struct M5Coef { T d, kappa, mass, c0; };

template <typename V, typename T> __device__ __forceinline__ V v_axpy(T a, V x, V y)      // a x + y
{
    V r;
    r.x = fma(a, x.x, y.x); r.y = fma(a, x.y, y.y);
    if constexpr (sizeof(V) == 16 && sizeof(T) == 4) { r.z = fma(a, x.z, y.z); r.w = fma(a, x.w, y.w); }
    return r;
}
template <typename V, typename T> __device__ __forceinline__ V v_scale(T a, V x)
{
    V r;
    r.x = a * x.x; r.y = a * x.y;
    if constexpr (sizeof(V) == 16 && sizeof(T) == 4) { r.z = a * x.z; r.w = a * x.w; }
    return r;
}
template <typename V> __device__ __forceinline__ V v_zero()
{
    V r;
    r.x = 0; r.y = 0;
    if constexpr (std::is_same<V, float4>::value) { r.z = 0; r.w = 0; }
    return r;
}

// chirality of the 128-bit vector v of a slice: true = spins 2,3 (the P_- components)
template <typename V> __device__ __forceinline__ bool is_minus(size_t v, int Lh)
{
    if constexpr (std::is_same<V, float4>::value) return ((v / (size_t)Lh) % 6) & 1;    // vector j: slots 2j, 2j+1 -> t = 0,1 | 2,3
    else return ((v / (size_t)Lh) % 12) >= 6;                                            // component k = spin*3 + colour
}

// OP 0: Mooee, 1: Mooee^{-1}; dagger swaps the chiralities (the matrices are real, the adjoint is the
// transpose, and the transpose of the P_+ block has the P_- stencil).  in == out is allowed (a thread
// reads all Ls values of its vector before it writes).  nblk half-field blocks of Ls slices each.
// EXACT: Ls == LSMAX, no predicates in the unrolled loops -- ptxas then issues all Ls loads of a thread
// back to back (with the runtime bound it interleaves them with the arithmetic of Mooee and loses
// memory-level parallelism: 342 us instead of 250 us on C4 fp32, r02).
template <typename V, typename T, int LSMAX, int OP, bool EXACT>
__global__ void __launch_bounds__(256)
s_op_kernel(const V *in, V *out, const size_t slice_vecs, const int nblk, const int Ls_arg, const int Lh,
            const bool dagger, const M5Coef<T> c)
{
    const int Ls = EXACT ? LSMAX : Ls_arg;
    const size_t n = slice_vecs * (size_t)nblk;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const size_t blk = t / slice_vecs, v = t % slice_vecs;
        const bool rev = is_minus<V>(v, Lh) != dagger;                // walk s downwards
        const size_t base = blk * slice_vecs * (size_t)Ls + v;
        const long long first = rev ? (long long)(Ls - 1) : 0, step = rev ? -1 : 1;
        V x[LSMAX];
#pragma unroll
        for (int i = 0; i < LSMAX; i++)
            if (i < Ls) x[i] = __ldcs(in + base + (size_t)(first + step * i) * slice_vecs);
        if constexpr (OP == 0) {
            V xlast = x[0];
#pragma unroll
            for (int i = 1; i < LSMAX; i++)
                if (i == Ls - 1) xlast = x[i];
#pragma unroll
            for (int i = LSMAX - 1; i >= 1; i--)
                if (i < Ls) x[i] = v_axpy<V, T>(c.d, x[i], v_scale<V, T>(T(-1), x[i - 1]));
            x[0] = v_axpy<V, T>(c.d, x[0], v_scale<V, T>(c.mass, xlast));
        } else {
            V acc = v_zero<V>();
#pragma unroll
            for (int i = 1; i < LSMAX; i++)
                if (i < Ls) acc = v_scale<V, T>(c.kappa, v_axpy<V, T>(T(1), acc, x[i]));
            x[0] = v_scale<V, T>(c.kappa * c.c0, v_axpy<V, T>(-c.mass, acc, x[0]));
#pragma unroll
            for (int i = 1; i < LSMAX; i++)
                if (i < Ls) x[i] = v_scale<V, T>(c.kappa, v_axpy<V, T>(T(1), x[i], x[i - 1]));
        }
#pragma unroll
        for (int i = 0; i < LSMAX; i++)
            if (i < Ls) __stcs(out + base + (size_t)(first + step * i) * slice_vecs, x[i]);
    }
}

// any Ls: the same recurrences with the vectors re-read from memory (two reads + one write; the second
// read mostly hits in L2).  in == out is NOT possible here, the caller goes through a copy.
template <typename V, typename T, int OP>
__global__ void __launch_bounds__(256)
s_op_generic_kernel(const V *__restrict__ in, V *__restrict__ out, const size_t slice_vecs, const int nblk, const int Ls,
                    const int Lh, const bool dagger, const M5Coef<T> c)
{
    const size_t n = slice_vecs * (size_t)nblk;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
        const size_t blk = t / slice_vecs, v = t % slice_vecs;
        const bool rev = is_minus<V>(v, Lh) != dagger;
        const size_t base = blk * slice_vecs * (size_t)Ls + v;
        const long long first = rev ? (long long)(Ls - 1) : 0, step = rev ? -1 : 1;
        auto at = [&](int i) { return base + (size_t)(first + step * i) * slice_vecs; };
        if constexpr (OP == 0) {
            V prev = in[at(Ls - 1)];
            V x0 = in[at(0)];
            out[at(0)] = v_axpy<V, T>(c.d, x0, v_scale<V, T>(c.mass, prev));
            prev = x0;
            for (int i = 1; i < Ls; i++) {
                const V xi = in[at(i)];
                out[at(i)] = v_axpy<V, T>(c.d, xi, v_scale<V, T>(T(-1), prev));
                prev = xi;
            }
        } else {
            V acc = v_zero<V>();
            for (int i = 1; i < Ls; i++) acc = v_scale<V, T>(c.kappa, v_axpy<V, T>(T(1), acc, in[at(i)]));
            V y = v_scale<V, T>(c.kappa * c.c0, v_axpy<V, T>(-c.mass, acc, in[at(0)]));
            out[at(0)] = y;
            for (int i = 1; i < Ls; i++) {
                y = v_scale<V, T>(c.kappa, v_axpy<V, T>(T(1), in[at(i)], y));
                out[at(i)] = y;
            }
        }
    }
}

template <typename V, typename T, int OP>
static int launch_s_op_t(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass, bool dagger,
                         cudaStream_t st)
{
    wait_for_exports(g, st, out, dwf_field_bytes(g, parity));
    const Lattice &lat = g->lat;
    const size_t vec_per_site = 96 * (size_t)g->prec / 4 / 16;                 // 6 (fp32) or 12 (fp64) vectors per site
    const size_t slice_vecs = (size_t)lat.Vh * vec_per_site;
    const int nblk = parity == DWF_FULL ? 2 : 1;
    const double d = 5.0 - M5;
    if (d == 0.0 || 1.0 + mass * pow(1.0 / d, lat.Ls) == 0.0) { set_error("Mooee is singular for M5 = %g, mass = %g", M5, mass); return DWF_ERR_INVALID_ARG; }
    M5Coef<T> c;
    c.d = (T)d; c.kappa = (T)(1.0 / d); c.mass = (T)mass; c.c0 = (T)(1.0 / (1.0 + mass * pow(1.0 / d, lat.Ls)));
    const size_t n = slice_vecs * (size_t)nblk;
    long long blocks = (long long)((n + 255) / 256);
    const long long cap = (long long)g->sm_count * 32;
    if (blocks > cap) blocks = cap;
    const V *pi = static_cast<const V *>(in);
    V *po = static_cast<V *>(out);
    const int Ls = lat.Ls;
#define DWF_SOP(LSM, EX) s_op_kernel<V, T, LSM, OP, EX><<<(unsigned)blocks, 256, 0, st>>>(pi, po, slice_vecs, nblk, Ls, lat.Lh, dagger, c)
    if (Ls == 8)       DWF_SOP(8, true);
    else if (Ls == 12) DWF_SOP(12, true);
    else if (Ls == 16) DWF_SOP(16, true);
    else if (Ls == 24) DWF_SOP(24, true);
    else if (Ls == 32) DWF_SOP(32, true);
    else if (Ls <= 8)  DWF_SOP(8, false);
    else if (Ls <= 16) DWF_SOP(16, false);
    else if (Ls <= 32) DWF_SOP(32, false);
#undef DWF_SOP
    else {
        if (in == out) { set_error("in-place fifth-dimension operators need Ls <= 32"); return DWF_ERR_UNSUPPORTED; }
        s_op_generic_kernel<V, T, OP><<<(unsigned)blocks, 256, 0, st>>>(pi, po, slice_vecs, nblk, Ls, lat.Lh, dagger, c);
    }
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

// op 0: Mooee, 1: Mooee^{-1}
static int launch_s_op(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass, int op, bool dagger,
                       cudaStream_t st)
{
    if (g->prec == DWF_F32)
        return op ? launch_s_op_t<float4, float, 1>(g, in, out, parity, M5, mass, dagger, st)
                  : launch_s_op_t<float4, float, 0>(g, in, out, parity, M5, mass, dagger, st);
    return op ? launch_s_op_t<double2, double, 1>(g, in, out, parity, M5, mass, dagger, st)
              : launch_s_op_t<double2, double, 0>(g, in, out, parity, M5, mass, dagger, st);
}

// ---------------------------------------------------------------------------------------------
// field algebra of the solver: 128-bit vectors, grid-stride, fp64 reductions in a fixed order
// ---------------------------------------------------------------------------------------------
template <typename V, typename T>
__global__ void __launch_bounds__(256)
axpby_kernel2(const T a, const V *x, const T b, const V *y, V *out, const size_t nvec)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x)
        out[i] = v_axpy<V, T>(a, x[i], v_scale<V, T>(b, y[i]));
}

// x += alpha p;  r -= alpha w;  partials[block] = sum |r|^2 of the block's elements (fp64)
template <typename V, typename T>
__global__ void __launch_bounds__(256)
cg_update_kernel(const T alpha, const V *__restrict__ p, const V *__restrict__ w, V *__restrict__ x, V *__restrict__ r,
                 const size_t nvec, double *__restrict__ partials)
{
    __shared__ double smem[32];
    double acc[1] = {0.0};
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        x[i] = v_axpy<V, T>(alpha, p[i], x[i]);
        const V rn = v_axpy<V, T>(-alpha, w[i], r[i]);
        r[i] = rn;
        acc[0] += (double)rn.x * rn.x + (double)rn.y * rn.y;
        if constexpr (std::is_same<V, float4>::value) acc[0] += (double)rn.z * rn.z + (double)rn.w * rn.w;
    }
    block_sum<1>(acc, smem);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc[0];
}

static int blas_blocks(const dwf_geometry *g, size_t nvec)
{
    long long b = (long long)((nvec + 255) / 256);
    const long long cap = g->reduce_blocks;
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

static int launch_axpby2(const dwf_geometry *g, double a, const void *x, double b, const void *y, void *out, size_t nreal,
                         cudaStream_t st)
{
    wait_for_exports(g, st, out, nreal * (size_t)g->prec);
    if (g->prec == DWF_F32) {
        const size_t nv = nreal / 4;
        axpby_kernel2<float4, float><<<blas_blocks(g, nv), 256, 0, st>>>((float)a, static_cast<const float4 *>(x), (float)b,
                                                                          static_cast<const float4 *>(y), static_cast<float4 *>(out), nv);
    } else {
        const size_t nv = nreal / 2;
        axpby_kernel2<double2, double><<<blas_blocks(g, nv), 256, 0, st>>>(a, static_cast<const double2 *>(x), b,
                                                                            static_cast<const double2 *>(y), static_cast<double2 *>(out), nv);
    }
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

// x += alpha p, r -= alpha w, *rr = |r|^2 (host, synchronises st)
static int cg_update(const dwf_geometry *g, double alpha, const void *p, const void *w, void *x, void *r, size_t nreal,
                     double *rr, cudaStream_t st)
{
    wait_for_exports(g, st);
    int nb;
    if (g->prec == DWF_F32) {
        const size_t nv = nreal / 4;
        nb = blas_blocks(g, nv);
        cg_update_kernel<float4, float><<<nb, 256, 0, st>>>((float)alpha, static_cast<const float4 *>(p), static_cast<const float4 *>(w),
                                                            static_cast<float4 *>(x), static_cast<float4 *>(r), nv, g->partials);
    } else {
        const size_t nv = nreal / 2;
        nb = blas_blocks(g, nv);
        cg_update_kernel<double2, double><<<nb, 256, 0, st>>>(alpha, static_cast<const double2 *>(p), static_cast<const double2 *>(w),
                                                              static_cast<double2 *>(x), static_cast<double2 *>(r), nv, g->partials);
    }
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    int rc = launch_final_sum(g, nb, st);
    if (rc) return rc;
    return fetch_reduction(g, st, 1, rr);
}

static int field_norm2(const dwf_geometry *g, const void *f, size_t nreal, double *out, cudaStream_t st)
{
    int rc = launch_norm2(g, f, nreal, st);
    if (rc) return rc;
    return fetch_reduction(g, st, 1, out);
}

// out = S in (dagger: S^dag in) on parity p; work = two half fields.  Four kernels.
static int schur_apply(const dwf_geometry *g, const void *in, void *out, int p, double M5, double mass, bool dagger, void *work,
                       cudaStream_t st)
{
    const size_t hb = dwf_field_bytes(g, DWF_EVEN);
    void *t = work, *u = static_cast<char *>(work) + hb;
    const int q = 1 - p;
    int rc;
    if ((rc = half_dhop(g, in, t, q, st, dagger))) return rc;                          // t_q = D_qp in
    if ((rc = launch_s_op(g, t, u, q, M5, mass, 1, dagger, st))) return rc;             // u_q = Mooee^{-1} t_q
    if ((rc = launch_s_op(g, in, out, p, M5, mass, 0, dagger, st))) return rc;          // out = Mooee in
    return half_dhop(g, u, out, p, st, dagger, out, 1.0, -0.25);                        // out = out - 1/4 D_pq u_q
}

}  // namespace dwf

using namespace dwf;

extern "C" {

static int check_s_args(const dwf_geometry *g, const void *in, const void *out, int parity, const char *who)
{
    if (!g || !in || !out || !parity_ok(parity)) { set_error("%s: bad argument", who); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(out)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    return DWF_OK;
}

int dwf_mooee(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass, int dagger, void *stream)
{
    int rc = check_s_args(g, in, out, parity, "dwf_mooee");
    if (rc) return rc;
    DeviceGuard guard(g->device);
    return launch_s_op(g, in, out, parity, M5, mass, 0, dagger != 0, static_cast<cudaStream_t>(stream));
}

int dwf_mooee_inv(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass, int dagger, void *stream)
{
    int rc = check_s_args(g, in, out, parity, "dwf_mooee_inv");
    if (rc) return rc;
    DeviceGuard guard(g->device);
    return launch_s_op(g, in, out, parity, M5, mass, 1, dagger != 0, static_cast<cudaStream_t>(stream));
}

int dwf_ddwf(const dwf_geometry *g, const void *in_full, void *out_full, double M5, double mass, int dagger, void *stream)
{
    int rc = check_s_args(g, in_full, out_full, DWF_FULL, "dwf_ddwf");
    if (rc) return rc;
    if (in_full == out_full) { set_error("dwf_ddwf: in-place application is not defined (in == out)"); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("dwf_ddwf: call dwf_load_gauge first"); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t hb = dwf_field_bytes(g, DWF_EVEN);
    const char *ie = static_cast<const char *>(in_full), *io = ie + hb;
    char *oe = static_cast<char *>(out_full), *oo = oe + hb;
    if ((rc = launch_s_op(g, in_full, out_full, DWF_FULL, M5, mass, 0, dagger != 0, st))) return rc;     // out = Mooee in
    if ((rc = half_dhop(g, ie, oo, DWF_ODD, st, dagger != 0, oo, 1.0, -0.5))) return rc;                 // out_o -= 1/2 D_oe in_e
    return half_dhop(g, io, oe, DWF_EVEN, st, dagger != 0, oe, 1.0, -0.5);                               // out_e -= 1/2 D_eo in_o
}

size_t dwf_schur_work_bytes(const dwf_geometry *g) { return g ? 2 * dwf_field_bytes(g, DWF_EVEN) : 0; }
size_t dwf_cg_work_bytes(const dwf_geometry *g) { return g ? 6 * dwf_field_bytes(g, DWF_EVEN) : 0; }

int dwf_schur(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass, int dagger, void *work,
              void *stream)
{
    int rc = check_s_args(g, in, out, parity, "dwf_schur");
    if (rc) return rc;
    if (parity == DWF_FULL || !work || !aligned16(work)) { set_error("dwf_schur: needs a half-field parity and a 16-byte aligned workspace"); return DWF_ERR_INVALID_ARG; }
    if (in == out) { set_error("dwf_schur: in-place application is not defined (in == out)"); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("dwf_schur: call dwf_load_gauge first"); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    return schur_apply(g, in, out, parity, M5, mass, dagger != 0, work, static_cast<cudaStream_t>(stream));
}

int dwf_axpby(const dwf_geometry *g, double a, const void *x, double b, const void *y, void *out, int parity, void *stream)
{
    if (!g || !x || !y || !out || !parity_ok(parity)) { set_error("dwf_axpby: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(x) || !aligned16(y) || !aligned16(out)) { set_error("dwf_axpby: field pointers must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    return launch_axpby2(g, a, x, b, y, out, dwf_field_bytes(g, parity) / (size_t)g->prec, static_cast<cudaStream_t>(stream));
}

int dwf_cg_schur(const dwf_geometry *g, const void *b, void *x, int parity, double M5, double mass, double tol, int max_iter,
                 void *work, int *iters_out, double *resid_out, void *stream)
{
    int rc = check_s_args(g, b, x, parity, "dwf_cg_schur");
    if (rc) return rc;
    if (parity == DWF_FULL || !work || !aligned16(work) || b == x || max_iter < 0 || !(tol >= 0.0)) {
        set_error("dwf_cg_schur: needs a half-field parity, a 16-byte aligned workspace, b != x, max_iter >= 0, tol >= 0");
        return DWF_ERR_INVALID_ARG;
    }
    if (!g->gauge_loaded) { set_error("dwf_cg_schur: call dwf_load_gauge first"); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t hb = dwf_field_bytes(g, DWF_EVEN), nreal = hb / (size_t)g->prec;
    char *wk = static_cast<char *>(work);
    void *r = wk, *p = wk + hb, *q = wk + 2 * hb, *w = wk + 3 * hb, *sw = wk + 4 * hb;      // sw: two half fields of the Schur kernels
    const bool dag = true;

    // conjugate gradients on the normal equations S^dag S x = S^dag b, x0 = 0
    double bb = 0.0, rr = 0.0, rr0;
    if ((rc = field_norm2(g, b, nreal, &bb, st))) return rc;
    DWF_CUDA_CHECK(cudaMemsetAsync(x, 0, hb, st));
    int it = 0;
    if (bb > 0.0) {
        if ((rc = schur_apply(g, b, r, parity, M5, mass, dag, sw, st))) return rc;           // r = S^dag b
        DWF_CUDA_CHECK(cudaMemcpyAsync(p, r, hb, cudaMemcpyDeviceToDevice, st));
        if ((rc = field_norm2(g, r, nreal, &rr, st))) return rc;
        rr0 = rr;
        while (it < max_iter && rr > tol * tol * rr0) {
            double qq = 0.0, rr_new = 0.0;
            if ((rc = schur_apply(g, p, q, parity, M5, mass, !dag, sw, st))) return rc;      // q = S p
            if ((rc = field_norm2(g, q, nreal, &qq, st))) return rc;
            if (!(qq > 0.0)) break;
            const double alpha = rr / qq;
            if ((rc = schur_apply(g, q, w, parity, M5, mass, dag, sw, st))) return rc;       // w = S^dag q
            if ((rc = cg_update(g, alpha, p, w, x, r, nreal, &rr_new, st))) return rc;       // x += alpha p, r -= alpha w
            it++;
            const double beta = rr_new / rr;
            rr = rr_new;
            if ((rc = launch_axpby2(g, 1.0, r, beta, p, p, nreal, st))) return rc;           // p = r + beta p
        }
    }
    // true residual |b - S x| / |b|
    double res = 0.0;
    if (bb > 0.0) {
        if ((rc = schur_apply(g, x, q, parity, M5, mass, !dag, sw, st))) return rc;
        if ((rc = launch_axpby2(g, 1.0, b, -1.0, q, q, nreal, st))) return rc;
        if ((rc = field_norm2(g, q, nreal, &res, st))) return rc;
        res = sqrt(res / bb);
    }
    if (iters_out) *iters_out = it;
    if (resid_out) *resid_out = res;
    return DWF_OK;
}

}  // extern "C"

// halo.cu -- time-direction domain decomposition of Dhop (PAPER.md L207 weak scaling, L223
// "near perfect overlap of communication and computation", L250 "face assembly": named there, no formulas;
// DESIGN.md reading #26).
//
// A rank owns a slab of the lattice along time (x3).  Its geometry has bc_time = DWF_OPEN_T: the stored
// wrapping time links are zero, so the ordinary Dhop kernels compute everything but the two face terms
//     first layer (x3 = 0):      (1 + gamma_t) U_t^dag(x - t) psi(x - t)     psi, U from the LOWER neighbour's last layer
//     last layer  (x3 = L3 - 1): (1 - gamma_t) U_t(x)         psi(x + t)     psi from the UPPER neighbour's first layer
// (Dhop^dagger: the projectors change places).  What travels between ranks is the projected half spinor, 12 reals
// per face site and slice: dwf_face_pack_t writes, for the upper neighbour, chi = U_t^dag(y) (1 + gamma_t) psi(y) of
// the slab's last layer (the link lives at the sender, so it is applied there) and, for the lower neighbour,
// (1 - gamma_t) psi(y) of the first layer; dwf_face_apply_t reconstructs the four spin components from the two
// received buffers, multiplies the upper face by U_t(x), and adds both to the slab's Dhop result.  The exchange
// itself (NCCL send / recv, or a copy when a rank is its own neighbour) is plumbing outside this library
// (paper_2203_06777_b200/dist.py) and runs while the bulk Dhop kernel computes.
// Face buffer: complex[s][row2][k6][h], k6 = alpha*3 + colour (alpha = 0, 1 the half-spinor component),
// row2 = x1 + L1*x2, h = x0 >> 1 of the face site (same h for the site on either side of the cut).
#include "complex_ops.cuh"
#include "dwf_internal.cuh"

namespace dwf {

template <typename T> struct FaceTypes;
template <> struct FaceTypes<float>  { using C = float2;  };
template <> struct FaceTypes<double> { using C = double2; };

// psi[spin][colour] of device site (s, row, h) of a half field
template <typename T>
__device__ __forceinline__ void load_site(const T *field, const Lattice &lat, long long nrow, int s, long long row, int h,
                                          typename FaceTypes<T>::C (&psi)[4][3])
{
    if constexpr (sizeof(T) == 4) {
        const float4 *v = reinterpret_cast<const float4 *>(field) + ((long long)s * nrow + row) * 6 * lat.Lh + h;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const float4 a = v[(2 * c) * lat.Lh], b = v[(2 * c + 1) * lat.Lh];     // (re0, re1, im0, im1), (re2, re3, im2, im3)
            psi[0][c] = make_float2(a.x, a.z); psi[1][c] = make_float2(a.y, a.w);
            psi[2][c] = make_float2(b.x, b.z); psi[3][c] = make_float2(b.y, b.w);
        }
    } else {
        const double2 *v = reinterpret_cast<const double2 *>(field) + ((long long)s * nrow + row) * 12 * lat.Lh + h;
#pragma unroll
        for (int sp = 0; sp < 4; sp++)
#pragma unroll
            for (int c = 0; c < 3; c++) psi[sp][c] = v[(sp * 3 + c) * lat.Lh];
    }
}

template <typename T>
__device__ __forceinline__ void store_site(T *field, const Lattice &lat, long long nrow, int s, long long row, int h,
                                           const typename FaceTypes<T>::C (&psi)[4][3])
{
    if constexpr (sizeof(T) == 4) {
        float4 *v = reinterpret_cast<float4 *>(field) + ((long long)s * nrow + row) * 6 * lat.Lh + h;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            v[(2 * c) * lat.Lh] = make_float4(psi[0][c].x, psi[1][c].x, psi[0][c].y, psi[1][c].y);
            v[(2 * c + 1) * lat.Lh] = make_float4(psi[2][c].x, psi[3][c].x, psi[2][c].y, psi[3][c].y);
        }
    } else {
        double2 *v = reinterpret_cast<double2 *>(field) + ((long long)s * nrow + row) * 12 * lat.Lh + h;
#pragma unroll
        for (int sp = 0; sp < 4; sp++)
#pragma unroll
            for (int c = 0; c < 3; c++) v[(sp * 3 + c) * lat.Lh] = psi[sp][c];
    }
}

template <typename C> __device__ __forceinline__ C c_add(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C c_sub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
// a + u * h  and  a + conj(u) * h
template <typename C> __device__ __forceinline__ C c_mac(C a, C u, C h)
{
    C r; r.x = fma(u.x, h.x, fma(-u.y, h.y, a.x)); r.y = fma(u.x, h.y, fma(u.y, h.x, a.y)); return r;
}
template <typename C> __device__ __forceinline__ C c_macc(C a, C u, C h)
{
    C r; r.x = fma(u.x, h.x, fma(u.y, h.y, a.x)); r.y = fma(u.x, h.y, fma(-u.y, h.x, a.y)); return r;
}

// tlink_top[q]: U_t(y) of the slab's last-layer sites y of parity q, complex[row2][9][h] (k = a*3 + b), WITHOUT
// boundary sign or zeroing (the packed gauge sets have the wrapping links zeroed / sign-folded)
template <typename T>
__global__ void __launch_bounds__(256)
tlink_pack_kernel(const T *__restrict__ U, T *__restrict__ top_even, T *__restrict__ top_odd, const Lattice lat)
{
    const long long nface = (long long)lat.L[0] * lat.L[1] * lat.L[2];        // lexicographic sites of the last layer
    const long long n = nface * 9;
    const int x3 = lat.L[3] - 1;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(e % 9);
        long long f = e / 9;
        const int x0 = (int)(f % lat.L[0]);
        const long long row2 = f / lat.L[0];
        const int x1 = (int)(row2 % lat.L[1]), x2 = (int)(row2 / lat.L[1]);
        const int par = (x0 + x1 + x2 + x3) & 1;
        const long long site = f + nface * x3;
        const T *u = U + ((site * 4 + 3) * 9 + k) * 2;
        T *dst = (par ? top_odd : top_even) + ((row2 * 9 + k) * lat.Lh + (x0 >> 1)) * 2;
        dst[0] = u[0];
        dst[1] = u[1];
    }
}

// one thread per (s, row2, h): both faces of the input half field (parity q)
template <typename T>
__global__ void __launch_bounds__(128)
face_pack_kernel(const T *__restrict__ in, const T *__restrict__ tlink_q, T *__restrict__ send_down, T *__restrict__ send_up,
                 const Lattice lat, const bool dagger)
{
    using C = typename FaceTypes<T>::C;
    const long long nrow2 = (long long)lat.L[1] * lat.L[2], nrow = nrow2 * lat.L[3];
    const long long n = (long long)lat.Ls * nrow2 * lat.Lh;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const int h = (int)(e % lat.Lh);
        const long long row2 = (e / lat.Lh) % nrow2;
        const int s = (int)(e / (lat.Lh * nrow2));
        C *dn = reinterpret_cast<C *>(send_down) + ((long long)s * nrow2 + row2) * 6 * lat.Lh + h;
        C *up = reinterpret_cast<C *>(send_up) + ((long long)s * nrow2 + row2) * 6 * lat.Lh + h;
        C psi[4][3];
        // first layer -> lower neighbour: upper components of (1 - gamma_t) psi  (dagger: 1 + gamma_t)
        load_site<T>(in, lat, nrow, s, row2, h, psi);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            dn[(0 * 3 + c) * lat.Lh] = dagger ? c_add(psi[0][c], psi[2][c]) : c_sub(psi[0][c], psi[2][c]);
            dn[(1 * 3 + c) * lat.Lh] = dagger ? c_add(psi[1][c], psi[3][c]) : c_sub(psi[1][c], psi[3][c]);
        }
        // last layer -> upper neighbour: chi = U_t^dag(y) (1 + gamma_t) psi(y), upper components  (dagger: 1 - gamma_t)
        load_site<T>(in, lat, nrow, s, row2 + nrow2 * (lat.L[3] - 1), h, psi);
        const C *u = reinterpret_cast<const C *>(tlink_q) + row2 * 9 * lat.Lh + h;
        C hh[2][3];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            hh[0][c] = dagger ? c_sub(psi[0][c], psi[2][c]) : c_add(psi[0][c], psi[2][c]);
            hh[1][c] = dagger ? c_sub(psi[1][c], psi[3][c]) : c_add(psi[1][c], psi[3][c]);
        }
#pragma unroll
        for (int a = 0; a < 3; a++) {
            C x0, x1;
            x0.x = x0.y = x1.x = x1.y = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const C ub = u[(b * 3 + a) * lat.Lh];                 // (U^dag)_ab = conj(U_ba)
                x0 = c_macc(x0, ub, hh[0][b]);
                x1 = c_macc(x1, ub, hh[1][b]);
            }
            up[(0 * 3 + a) * lat.Lh] = x0;
            up[(1 * 3 + a) * lat.Lh] = x1;
        }
    }
}

// one thread per (s, row2, h): adds the two face terms to the output half field (parity p)
template <typename T>
__global__ void __launch_bounds__(128)
face_apply_kernel(const T *__restrict__ recv_lo, const T *__restrict__ recv_hi, const T *__restrict__ tlink_p, T *__restrict__ out,
                  const Lattice lat, const bool dagger, const T sign_lo, const T sign_hi)
{
    using C = typename FaceTypes<T>::C;
    const long long nrow2 = (long long)lat.L[1] * lat.L[2], nrow = nrow2 * lat.L[3];
    const long long n = (long long)lat.Ls * nrow2 * lat.Lh;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const int h = (int)(e % lat.Lh);
        const long long row2 = (e / lat.Lh) % nrow2;
        const int s = (int)(e / (lat.Lh * nrow2));
        const C *lo = reinterpret_cast<const C *>(recv_lo) + ((long long)s * nrow2 + row2) * 6 * lat.Lh + h;
        const C *hi = reinterpret_cast<const C *>(recv_hi) + ((long long)s * nrow2 + row2) * 6 * lat.Lh + h;
        C psi[4][3];
        // first layer: backward hop, (1 + gamma_t): r2 = +h0, r3 = +h1   (dagger, 1 - gamma_t: r2 = -h0, r3 = -h1)
        load_site<T>(out, lat, nrow, s, row2, h, psi);
        const T lw = dagger ? -sign_lo : sign_lo;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const C x0 = lo[(0 * 3 + c) * lat.Lh], x1 = lo[(1 * 3 + c) * lat.Lh];
            psi[0][c].x = fma(sign_lo, x0.x, psi[0][c].x); psi[0][c].y = fma(sign_lo, x0.y, psi[0][c].y);
            psi[1][c].x = fma(sign_lo, x1.x, psi[1][c].x); psi[1][c].y = fma(sign_lo, x1.y, psi[1][c].y);
            psi[2][c].x = fma(lw, x0.x, psi[2][c].x); psi[2][c].y = fma(lw, x0.y, psi[2][c].y);
            psi[3][c].x = fma(lw, x1.x, psi[3][c].x); psi[3][c].y = fma(lw, x1.y, psi[3][c].y);
        }
        store_site<T>(out, lat, nrow, s, row2, h, psi);
        // last layer: forward hop, chi = U_t(x) h, (1 - gamma_t): r2 = -chi0, r3 = -chi1   (dagger: +)
        const long long rtop = row2 + nrow2 * (lat.L[3] - 1);
        load_site<T>(out, lat, nrow, s, rtop, h, psi);
        const C *u = reinterpret_cast<const C *>(tlink_p) + row2 * 9 * lat.Lh + h;
        C hh[2][3];
#pragma unroll
        for (int c = 0; c < 3; c++) { hh[0][c] = hi[(0 * 3 + c) * lat.Lh]; hh[1][c] = hi[(1 * 3 + c) * lat.Lh]; }
        const T uw = dagger ? sign_hi : -sign_hi;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            C x0, x1;
            x0.x = x0.y = x1.x = x1.y = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const C ub = u[(a * 3 + b) * lat.Lh];
                x0 = c_mac(x0, ub, hh[0][b]);
                x1 = c_mac(x1, ub, hh[1][b]);
            }
            psi[0][a].x = fma(sign_hi, x0.x, psi[0][a].x); psi[0][a].y = fma(sign_hi, x0.y, psi[0][a].y);
            psi[1][a].x = fma(sign_hi, x1.x, psi[1][a].x); psi[1][a].y = fma(sign_hi, x1.y, psi[1][a].y);
            psi[2][a].x = fma(uw, x0.x, psi[2][a].x); psi[2][a].y = fma(uw, x0.y, psi[2][a].y);
            psi[3][a].x = fma(uw, x1.x, psi[3][a].x); psi[3][a].y = fma(uw, x1.y, psi[3][a].y);
        }
        store_site<T>(out, lat, nrow, s, rtop, h, psi);
    }
}

static int face_grid(const dwf_geometry *g)
{
    const long long n = (long long)g->lat.Ls * g->lat.L[1] * g->lat.L[2] * g->lat.Lh;
    long long b = (n + 127) / 128;
    const long long cap = (long long)g->sm_count * 16;
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

int launch_pack_tlinks(const dwf_geometry *g, const void *U_dev, cudaStream_t st)
{
    const long long n = (long long)g->lat.L[0] * g->lat.L[1] * g->lat.L[2] * 9;
    const int grid = (int)((n + 255) / 256 < 4096 ? (n + 255) / 256 : 4096);
    if (g->prec == DWF_F32)
        tlink_pack_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float *>(U_dev), static_cast<float *>(g->tlink_top[0]),
                                                      static_cast<float *>(g->tlink_top[1]), g->lat);
    else
        tlink_pack_kernel<double><<<grid, 256, 0, st>>>(static_cast<const double *>(U_dev), static_cast<double *>(g->tlink_top[0]),
                                                       static_cast<double *>(g->tlink_top[1]), g->lat);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

}  // namespace dwf

using namespace dwf;

extern "C" {

size_t dwf_face_bytes(const dwf_geometry *g)
{
    if (!g) return 0;
    return (size_t)g->lat.Ls * g->lat.L[1] * g->lat.L[2] * g->lat.Lh * 12 * (size_t)g->prec;
}

int dwf_face_pack_t(const dwf_geometry *g, const void *in, int parity_in, int dagger, void *send_down, void *send_up, void *stream)
{
    if (!g || !in || !send_down || !send_up || (parity_in != DWF_EVEN && parity_in != DWF_ODD)) { set_error("dwf_face_pack_t: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(send_down) || !aligned16(send_up)) { set_error("dwf_face_pack_t: pointers must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("dwf_face_pack_t: call dwf_load_gauge first"); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (g->prec == DWF_F32)
        face_pack_kernel<float><<<face_grid(g), 128, 0, st>>>(static_cast<const float *>(in), static_cast<const float *>(g->tlink_top[parity_in]),
                                                             static_cast<float *>(send_down), static_cast<float *>(send_up), g->lat, dagger != 0);
    else
        face_pack_kernel<double><<<face_grid(g), 128, 0, st>>>(static_cast<const double *>(in), static_cast<const double *>(g->tlink_top[parity_in]),
                                                              static_cast<double *>(send_down), static_cast<double *>(send_up), g->lat, dagger != 0);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

int dwf_face_apply_t(const dwf_geometry *g, const void *recv_lo, const void *recv_hi, double sign_lo, double sign_hi, void *out,
                     int parity_out, int dagger, void *stream)
{
    if (!g || !recv_lo || !recv_hi || !out || (parity_out != DWF_EVEN && parity_out != DWF_ODD)) { set_error("dwf_face_apply_t: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(out) || !aligned16(recv_lo) || !aligned16(recv_hi)) { set_error("dwf_face_apply_t: pointers must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("dwf_face_apply_t: call dwf_load_gauge first"); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    wait_for_exports(g, st, out, dwf_field_bytes(g, parity_out));
    if (g->prec == DWF_F32)
        face_apply_kernel<float><<<face_grid(g), 128, 0, st>>>(static_cast<const float *>(recv_lo), static_cast<const float *>(recv_hi),
                                                              static_cast<const float *>(g->tlink_top[parity_out]), static_cast<float *>(out), g->lat,
                                                              dagger != 0, (float)sign_lo, (float)sign_hi);
    else
        face_apply_kernel<double><<<face_grid(g), 128, 0, st>>>(static_cast<const double *>(recv_lo), static_cast<const double *>(recv_hi),
                                                               static_cast<const double *>(g->tlink_top[parity_out]), static_cast<double *>(out), g->lat,
                                                               dagger != 0, sign_lo, sign_hi);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

}  // extern "C"

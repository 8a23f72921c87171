// dhop.cu -- the direct (L1-cached) Dhop kernel (hot path rows a2-a6 of SURVEY.md section 8): the
// general path for every geometry and precision; dhop_staged.cu holds the fast fp32 path.
//
//   Dhop psi(x,s) = sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu,s) + (1+gamma_mu) U_mu^dag(x-mu) psi(x-mu,s) ]
//
// One thread owns one output 4D site and SC consecutive s-slices.  For each of the 8 legs it
//   (a2) computes the neighbour's site index (periodic wrap; checkerboard x0 rule),
//   (a3) loads the neighbour spinor (12 complex x SC, 128-bit loads) and projects it with
//        (1 -/+ gamma_mu) to a half spinor (2 spins x 3 colours),
//   (a4) loads the link for this leg ONCE and multiplies it into the SC half spinors,
//   (a5) reconstructs the lower two spin components and accumulates in registers,
// then writes the 12 x SC complex results with streaming stores.  Backward links are stored
// pre-daggered and carry the antiperiodic sign, so all 8 legs run the same mat-vec.
//
// Projection / reconstruction in the DeGrand-Rossi basis (derived from gamma (1 +/- gamma) =
// +/-(1 +/- gamma); rows 0,1 of (1 + e gamma_mu) psi are h0,h1, rows 2,3 follow from them):
//   mu=x: h0 = psi0 + e i psi3, h1 = psi1 + e i psi2, r2 = -e i h1, r3 = -e i h0
//   mu=y: h0 = psi0 - e   psi3, h1 = psi1 + e   psi2, r2 =  e   h1, r3 = -e   h0
//   mu=z: h0 = psi0 + e i psi2, h1 = psi1 - e i psi3, r2 = -e i h0, r3 =  e i h1
//   mu=t: h0 = psi0 + e   psi2, h1 = psi1 + e   psi3, r2 =  e   h0, r3 =  e   h1
// with e = -1 on the forward leg (x+mu) and e = +1 on the backward leg (x-mu).
#include "complex_ops.cuh"
#include "dwf_internal.cuh"

namespace dwf {

// element offset of component c of a site inside a row block stored as [c/2][h][c&1]; `W0` = Lh,
// the pointer it is added to already points at (component 0, this site) = row base + 2*h
__device__ __forceinline__ int pair_off(int c, int W0) { return (c >> 1) * 2 * W0 + (c & 1); }

// gauge storage: complex[row][f/2][h][f&1], f = leg*9 + a*3+b; `site_links` points at f = 0 of this site
template <typename T, int LEG>
__device__ __forceinline__ void load_link(const typename CxT<T>::type *site_links, int W0, typename CxT<T>::type (&U)[9])
{
#pragma unroll
    for (int v = 0; v < 9; v++) U[v] = __ldg(site_links + pair_off(LEG * 9 + v, W0));
}

// one leg: acc += reconstruct( U * project(psi_neighbour) )
template <typename T, int SC, int MU, bool FWD, bool FIRST, int LEG>
__device__ __forceinline__ void dhop_leg(typename CxT<T>::type (&acc)[12][SC],
                                         const typename CxT<T>::type *__restrict__ nb,  // neighbour, component 0
                                         int W0,                                        // Lh
                                         const typename CxT<T>::type *__restrict__ site_links)
{
    using C = typename CxT<T>::type;
    C psi[12][SC];
    if constexpr (sizeof(T) == 8) {
#pragma unroll
        for (int k = 0; k < 12; k++) load_cx<SC>(nb + k * W0, psi[k]);      // fp64 fields: complex[..][k][h]
    } else {
        // fp32 fields store spin pairs (pack.cu): slot 4c + t -> (re|im of spins 0,1 | 2,3)
        C q[12][SC];
#pragma unroll
        for (int k = 0; k < 12; k++) load_cx<SC>(nb + pair_off(k, W0), q[k]);
#pragma unroll
        for (int j = 0; j < SC; j++)
#pragma unroll
            for (int c = 0; c < 3; c++) {
                psi[0 + c][j] = C{q[4 * c + 0][j].x, q[4 * c + 1][j].x};
                psi[3 + c][j] = C{q[4 * c + 0][j].y, q[4 * c + 1][j].y};
                psi[6 + c][j] = C{q[4 * c + 2][j].x, q[4 * c + 3][j].x};
                psi[9 + c][j] = C{q[4 * c + 2][j].y, q[4 * c + 3][j].y};
            }
    }
    C U[9];
    load_link<T, LEG>(site_links, W0, U);

#pragma unroll
    for (int j = 0; j < SC; j++) {
        C h0[3], h1[3];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const C p0 = psi[0 + c][j], p1 = psi[3 + c][j], p2 = psi[6 + c][j], p3 = psi[9 + c][j];
            if constexpr (MU == 0) {
                h0[c] = FWD ? csubi(p0, p3) : caddi(p0, p3);
                h1[c] = FWD ? csubi(p1, p2) : caddi(p1, p2);
            } else if constexpr (MU == 1) {
                h0[c] = FWD ? cadd(p0, p3) : csub(p0, p3);
                h1[c] = FWD ? csub(p1, p2) : cadd(p1, p2);
            } else if constexpr (MU == 2) {
                h0[c] = FWD ? csubi(p0, p2) : caddi(p0, p2);
                h1[c] = FWD ? caddi(p1, p3) : csubi(p1, p3);
            } else {
                h0[c] = FWD ? csub(p0, p2) : cadd(p0, p2);
                h1[c] = FWD ? csub(p1, p3) : cadd(p1, p3);
            }
        }
#pragma unroll
        for (int a = 0; a < 3; a++) {
            C x0 = cmul(U[3 * a], h0[0]);
            x0 = cmac(x0, U[3 * a + 1], h0[1]);
            x0 = cmac(x0, U[3 * a + 2], h0[2]);
            C x1 = cmul(U[3 * a], h1[0]);
            x1 = cmac(x1, U[3 * a + 1], h1[1]);
            x1 = cmac(x1, U[3 * a + 2], h1[2]);
            // rows 2,3 as multiples of x0/x1: value = sgn * (i?) * x
            if constexpr (FIRST) {
                acc[0 + a][j] = x0;
                acc[3 + a][j] = x1;
                if constexpr (MU == 0) {
                    acc[6 + a][j] = FWD ? cmuli(x1) : cmulni(x1);
                    acc[9 + a][j] = FWD ? cmuli(x0) : cmulni(x0);
                } else if constexpr (MU == 1) {
                    acc[6 + a][j] = FWD ? cneg(x1) : x1;
                    acc[9 + a][j] = FWD ? x0 : cneg(x0);
                } else if constexpr (MU == 2) {
                    acc[6 + a][j] = FWD ? cmuli(x0) : cmulni(x0);
                    acc[9 + a][j] = FWD ? cmulni(x1) : cmuli(x1);
                } else {
                    acc[6 + a][j] = FWD ? cneg(x0) : x0;
                    acc[9 + a][j] = FWD ? cneg(x1) : x1;
                }
            } else {
                acc[0 + a][j] = cadd(acc[0 + a][j], x0);
                acc[3 + a][j] = cadd(acc[3 + a][j], x1);
                if constexpr (MU == 0) {
                    acc[6 + a][j] = FWD ? caddi(acc[6 + a][j], x1) : csubi(acc[6 + a][j], x1);
                    acc[9 + a][j] = FWD ? caddi(acc[9 + a][j], x0) : csubi(acc[9 + a][j], x0);
                } else if constexpr (MU == 1) {
                    acc[6 + a][j] = FWD ? csub(acc[6 + a][j], x1) : cadd(acc[6 + a][j], x1);
                    acc[9 + a][j] = FWD ? cadd(acc[9 + a][j], x0) : csub(acc[9 + a][j], x0);
                } else if constexpr (MU == 2) {
                    acc[6 + a][j] = FWD ? caddi(acc[6 + a][j], x0) : csubi(acc[6 + a][j], x0);
                    acc[9 + a][j] = FWD ? csubi(acc[9 + a][j], x1) : caddi(acc[9 + a][j], x1);
                } else {
                    acc[6 + a][j] = FWD ? csub(acc[6 + a][j], x0) : cadd(acc[6 + a][j], x0);
                    acc[9 + a][j] = FWD ? csub(acc[9 + a][j], x1) : cadd(acc[9 + a][j], x1);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// direct kernel: neighbours are read straight from global memory (L1/L2 catch the reuse).
// in/out are half fields pair[s][row][k/2][h][k&1] (slot meaning: pack.cu); out has parity `parity_out`, in the opposite parity.
// One thread = one output site and one s-slice.
// ---------------------------------------------------------------------------------------------
// DAG: Dhop^dagger -- the projectors (1 - gamma) and (1 + gamma) change places
// AXPY: out = a x + b Dhop in, x a half field of the output parity read at the thread's own site (x may
// be out: every thread reads its x before it writes)
template <typename T, int MAXT, int MINB, bool DAG, bool AXPY>
__global__ void __launch_bounds__(MAXT, MINB)
dhop_direct_kernel(const typename CxT<T>::type *__restrict__ in, typename CxT<T>::type *out,
                   const T *__restrict__ gset, const int4 *__restrict__ tiles, const Lattice lat,
                   const Tiling til, const int parity_out, const typename CxT<T>::type *xf, const T ca, const T cb)
{
    using C = typename CxT<T>::type;
    constexpr int SC = 1;
    const int nsh = til.sh[0] + til.sh[1] + til.sh[2] + til.sh[3];
    const int tid = threadIdx.x;
    const int ls = tid & ((1 << nsh) - 1);
    const int s = (blockIdx.x % til.ncg) * til.cpc + (tid >> nsh);
    const int4 org = tiles[blockIdx.x / til.ncg];

    int l = ls;
    const int c0 = org.x + (l & ((1 << til.sh[0]) - 1)); l >>= til.sh[0];
    const int x1 = org.y + (l & ((1 << til.sh[1]) - 1)); l >>= til.sh[1];
    const int x2 = org.z + (l & ((1 << til.sh[2]) - 1)); l >>= til.sh[2];
    const int x3 = org.w + l;

    const int L1 = lat.L[1], L2 = lat.L[2], L3 = lat.L[3];
    const int W0 = lat.Lh;                           // row length in field sites
    const long long Vh = lat.Vh;

    // a row (lattice line along x0) is a block of 12*W0 complex: [k/2][h][k&1]
    const long long row = x1 + L1 * (x2 + (long long)L2 * x3);
    const long long rs = 12 * W0;                    // complex elements per row
    constexpr int SS = sizeof(T) == 4 ? 2 : 1;       // complex elements between consecutive sites of a component plane
    const long long own = row * rs + SS * c0;

    // neighbour element offsets (component 0)
    const int r = (x1 + x2 + x3 + parity_out) & 1;          // x0 = 2*c0 + r
    int hp = c0 + r;       if (hp == W0) hp = 0;
    int hm = c0 - 1 + r;   if (hm < 0) hm = W0 - 1;
    const long long n0p = row * rs + SS * hp;
    const long long n0m = row * rs + SS * hm;
    const long long s1 = rs, s2 = rs * L1, s3 = rs * L1 * L2;
    const long long n1p = own + (x1 + 1 == L1 ? -(L1 - 1) * s1 : s1);
    const long long n1m = own + (x1 == 0 ? (L1 - 1) * s1 : -s1);
    const long long n2p = own + (x2 + 1 == L2 ? -(L2 - 1) * s2 : s2);
    const long long n2m = own + (x2 == 0 ? (L2 - 1) * s2 : -s2);
    const long long n3p = own + (x3 + 1 == L3 ? -(L3 - 1) * s3 : s3);
    const long long n3m = own + (x3 == 0 ? (L3 - 1) * s3 : -s3);

    const C *base = in + (size_t)s * 12 * (size_t)Vh;
    const C *gl = reinterpret_cast<const C *>(gset) + (size_t)row * 72 * W0 + 2 * c0;   // this site's links

    C acc[12][SC];
    dhop_leg<T, SC, 0, true != DAG, true, 0>(acc, base + n0p, W0, gl);
    dhop_leg<T, SC, 0, false != DAG, false, 1>(acc, base + n0m, W0, gl);
    dhop_leg<T, SC, 1, true != DAG, false, 2>(acc, base + n1p, W0, gl);
    dhop_leg<T, SC, 1, false != DAG, false, 3>(acc, base + n1m, W0, gl);
    dhop_leg<T, SC, 2, true != DAG, false, 4>(acc, base + n2p, W0, gl);
    dhop_leg<T, SC, 2, false != DAG, false, 5>(acc, base + n2m, W0, gl);
    dhop_leg<T, SC, 3, true != DAG, false, 6>(acc, base + n3p, W0, gl);
    dhop_leg<T, SC, 3, false != DAG, false, 7>(acc, base + n3m, W0, gl);

    C *o = out + (size_t)s * 12 * (size_t)Vh + (size_t)own;
    const C *xo = AXPY ? xf + (size_t)s * 12 * (size_t)Vh + (size_t)own : nullptr;
    if constexpr (sizeof(T) == 8) {
        if constexpr (AXPY) {
#pragma unroll
            for (int k = 0; k < 12; k++) {
                const C xv = xo[k * W0];
                acc[k][0].x = fma(cb, acc[k][0].x, ca * xv.x);
                acc[k][0].y = fma(cb, acc[k][0].y, ca * xv.y);
            }
        }
#pragma unroll
        for (int k = 0; k < 12; k++) store_cx<SC>(o + k * W0, acc[k]);
    } else {
#pragma unroll
        for (int c = 0; c < 3; c++) {
            C q[4][SC];
#pragma unroll
            for (int j = 0; j < SC; j++) {
                q[0][j] = C{acc[0 + c][j].x, acc[3 + c][j].x};
                q[1][j] = C{acc[0 + c][j].y, acc[3 + c][j].y};
                q[2][j] = C{acc[6 + c][j].x, acc[9 + c][j].x};
                q[3][j] = C{acc[6 + c][j].y, acc[9 + c][j].y};
            }
            if constexpr (AXPY) {
#pragma unroll
                for (int t = 0; t < 4; t++) {
                    const C xv = xo[pair_off(4 * c + t, W0)];
                    q[t][0].x = fmaf(cb, q[t][0].x, ca * xv.x);
                    q[t][0].y = fmaf(cb, q[t][0].y, ca * xv.y);
                }
            }
#pragma unroll
            for (int t = 0; t < 4; t++) store_cx<SC>(o + pair_off(4 * c + t, W0), q[t]);
        }
    }
}

template <typename T, int MAXT, int MINB, bool DAG, bool AXPY>
static int launch_direct(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st,
                         const void *x, double a, double b)
{
    using C = typename CxT<T>::type;
    const Tiling &til = g->tiling_cb;
    if (til.threads > MAXT) {
        set_error("tile of %d threads exceeds kernel limit %d", til.threads, MAXT);
        return DWF_ERR_UNSUPPORTED;
    }
    dim3 grid((unsigned)(til.ntiles * til.ncg)), block((unsigned)til.threads);
    dhop_direct_kernel<T, MAXT, MINB, DAG, AXPY><<<grid, block, 0, st>>>(
        static_cast<const C *>(in), static_cast<C *>(out), static_cast<const T *>(g->gauge[parity_out]),
        g->tiles_cb, g->lat, til, parity_out, static_cast<const C *>(x), (T)a, (T)b);
    count_launch();
    DWF_CUDA_CHECK(cudaGetLastError());
    return DWF_OK;
}

// parity_out: DWF_EVEN (DhopEO) or DWF_ODD (DhopOE); axpy_x != nullptr: out = a x + b Dhop in
int launch_dhop_direct(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st, bool dagger,
                       const void *axpy_x, double a, double b)
{
    if (g->prec == DWF_F32) {
        if (axpy_x)
            return dagger ? launch_direct<float, 256, 3, true, true>(g, in, out, parity_out, st, axpy_x, a, b)
                          : launch_direct<float, 256, 3, false, true>(g, in, out, parity_out, st, axpy_x, a, b);
        return dagger ? launch_direct<float, 256, 3, true, false>(g, in, out, parity_out, st, nullptr, 0, 0)
                      : launch_direct<float, 256, 3, false, false>(g, in, out, parity_out, st, nullptr, 0, 0);
    }
    if (axpy_x)
        return dagger ? launch_direct<double, 256, 2, true, true>(g, in, out, parity_out, st, axpy_x, a, b)
                      : launch_direct<double, 256, 2, false, true>(g, in, out, parity_out, st, axpy_x, a, b);
    return dagger ? launch_direct<double, 256, 2, true, false>(g, in, out, parity_out, st, nullptr, 0, 0)
                  : launch_direct<double, 256, 2, false, false>(g, in, out, parity_out, st, nullptr, 0, 0);
}

}  // namespace dwf

// dhop_staged64.cu -- the fp64 TMA-staged Dhop kernel for sm_100a: link-stationary with the links of
// a site split by COLOUR COLUMN over three threads.
//
//   Dhop psi(x,s) = sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu,s) + (1+gamma_mu) U_mu^dag(x-mu) psi(x-mu,s) ]
//
// In fp64 the 8 links of a site are 288 registers, so the fp32 scheme (dhop_staged.cu: one thread per
// site keeps them all) does not fit.  Here thread (site, c) keeps column c of every link -- the three
// numbers U_ac, a = 0..2, of each of the 8 legs: 24 complex = 96 registers -- and needs only colour c of
// the neighbour spinors: it loads 4 complex per leg, projects them to h_0c, h_1c, forms the partial
// products U_ac h_alpha,c and reconstructs / accumulates them into 12 partial sums exactly as the
// full kernel does (projection, SU(3) product and reconstruction are linear, so the sum over c can
// wait until all 8 legs are done).  After the legs the three threads of a site exchange partial sums
// through shared memory (each owns 4 of the 12 output components), add them in a fixed order and
// store.  Threads are colour-major (a warp = one colour of 32 consecutive sites), so every LDS / STG is
// conflict-free and coalesced and there is no divergence.
// Everything else follows dhop_staged.cu: a producer warpgroup (setmaxnreg) issues 5-D bulk tensor
// copies (TMA) of the input slice -- rows box + 6 faces -- into a two-stage shared-memory ring with
// full / empty mbarriers; consumers walk all Ls slices of a tile with their link columns in registers.
// Layouts (pack.cu): spinor complex[s][row][k][h], k = spin*3 + colour (one plane per component:
// consecutive sites are consecutive 128-bit words); links
// complex[row][f/2][h][f&1], f = leg*9 + a*3 + b.
#include <vector>

#include "complex_ops.cuh"
#include "dwf_internal.cuh"
#include "tma.cuh"

namespace dwf {

PFN_tensorMapEncodeTiled get_tensor_map_encoder();      // dhop_staged.cu

struct Staged64Args {
    double2 *out;
    const double2 *gauge;    // gauge set of the output parity: [row][36 pairs][Lh][2]
    const int4 *tiles;       // origins (o1, o2, o3) of the row boxes, launch order
    int ntiles;
    int L1, L2, L3, Ls;
    int parity_out;
    const double2 *axpy_x;   // AXPY kernels: out = a x + b Dhop in (x on the output parity; may be out)
    double axpy_a, axpy_b;
};

template <int LH, int B1, int B2, int B3> struct Staged64Cfg {
    static constexpr int NROW_C = B1 * B2 * B3;
    static constexpr int T = LH * NROW_C;                        // output sites per tile
    static constexpr int TP = (T + 31) / 32 * 32;                // sites padded to whole warps: thread = colour * TP + site
    static constexpr int NGROUP = TP / 32;                       // 32-site groups = named barriers
    static constexpr int NWARP_C = 3 * NGROUP;
    static constexpr int NTC = (3 * TP + 127) / 128 * 128;       // consumer threads (whole warpgroups)
    static constexpr int NT = 128 + NTC;
    static constexpr int ROWB = 12 * LH * 16;                    // bytes of one staged row
    static constexpr int R_X1M = NROW_C, R_X1P = R_X1M + B2 * B3, R_X2M = R_X1P + B2 * B3,
                         R_X2P = R_X2M + B1 * B3, R_X3M = R_X2P + B1 * B3, R_X3P = R_X3M + B1 * B2,
                         NROW_IN = R_X3P + B1 * B2;
    static constexpr int STAGE_BYTES = NROW_IN * ROWB;
    static constexpr int NSTAGE = 2;
    // exchange buffer: [parity of the step][destination colour][source slot][component j][site] complex
    static constexpr int RED_BYTES = 2 * 3 * 2 * 4 * TP * 16;
    static constexpr int TAIL = 64;                              // full[2], empty[2] mbarriers
    static constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + RED_BYTES + TAIL;
    static constexpr int PROD_REGS = 24;
    static constexpr int CONS_REGS_RAW = ((65536 - 128 * PROD_REGS) / NTC) / 8 * 8;
    static constexpr int CONS_REGS = CONS_REGS_RAW > 240 ? 240 : CONS_REGS_RAW;
    static_assert(ROWB % 128 == 0, "staged rows must keep TMA destinations 128-byte aligned");
    static_assert(SMEM_BYTES <= 232448, "tile too large for shared memory");
};

// one leg for colour c: acc += reconstruct( U[:, c] * project(psi)[c] ).  p0..p3 = colour c of the four
// spin components of the neighbour, U = (U_0c, U_1c, U_2c).  Signs as in dhop.cu (DeGrand-Rossi).
template <int MU, bool FWD>
__device__ __forceinline__ void leg64(double2 (&acc)[12], const double2 p0, const double2 p1, const double2 p2,
                                      const double2 p3, const double2 *__restrict__ U)
{
    double2 h0, h1;
    if constexpr (MU == 0) {
        h0 = FWD ? csubi(p0, p3) : caddi(p0, p3);
        h1 = FWD ? csubi(p1, p2) : caddi(p1, p2);
    } else if constexpr (MU == 1) {
        h0 = FWD ? cadd(p0, p3) : csub(p0, p3);
        h1 = FWD ? csub(p1, p2) : cadd(p1, p2);
    } else if constexpr (MU == 2) {
        h0 = FWD ? csubi(p0, p2) : caddi(p0, p2);
        h1 = FWD ? caddi(p1, p3) : csubi(p1, p3);
    } else {
        h0 = FWD ? csub(p0, p2) : cadd(p0, p2);
        h1 = FWD ? csub(p1, p3) : cadd(p1, p3);
    }
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const double2 x0 = cmul(U[a], h0), x1 = cmul(U[a], h1);
        acc[0 + a] = cadd(acc[0 + a], x0);
        acc[3 + a] = cadd(acc[3 + a], x1);
        if constexpr (MU == 0) {
            acc[6 + a] = FWD ? caddi(acc[6 + a], x1) : csubi(acc[6 + a], x1);
            acc[9 + a] = FWD ? caddi(acc[9 + a], x0) : csubi(acc[9 + a], x0);
        } else if constexpr (MU == 1) {
            acc[6 + a] = FWD ? csub(acc[6 + a], x1) : cadd(acc[6 + a], x1);
            acc[9 + a] = FWD ? cadd(acc[9 + a], x0) : csub(acc[9 + a], x0);
        } else if constexpr (MU == 2) {
            acc[6 + a] = FWD ? caddi(acc[6 + a], x0) : csubi(acc[6 + a], x0);
            acc[9 + a] = FWD ? csubi(acc[9 + a], x1) : caddi(acc[9 + a], x1);
        } else {
            acc[6 + a] = FWD ? csub(acc[6 + a], x0) : cadd(acc[6 + a], x0);
            acc[9 + a] = FWD ? csub(acc[9 + a], x1) : cadd(acc[9 + a], x1);
        }
    }
}

// consumer body for colour column C (compile-time: the colour of a warp is uniform)
template <int LH, int B1, int B2, int B3, bool DAG, bool AXPY, int C>
__device__ __forceinline__ void consume64(const Staged64Args &args, unsigned char *smem, const uint32_t full_base,
                                          const uint32_t empty_base, const int site, const int my_tiles)
{
    using Cfg = Staged64Cfg<LH, B1, B2, B3>;
    const bool active = site < Cfg::T;
    const int st = active ? site : 0;
    const int h = st % LH, row = st / LH;
    const int i1 = row % B1, i2 = (row / B1) % B2, i3 = row / (B1 * B2);
    const int lane = threadIdx.x & 31;

    // staged rows of the 8 neighbours (tile-invariant except the x0 pair)
    const int rc = row;
    const int r1p = (i1 + 1 < B1) ? rc + 1 : Cfg::R_X1P + i2 + B2 * i3;
    const int r1m = (i1 > 0) ? rc - 1 : Cfg::R_X1M + i2 + B2 * i3;
    const int r2p = (i2 + 1 < B2) ? rc + B1 : Cfg::R_X2P + i1 + B1 * i3;
    const int r2m = (i2 > 0) ? rc - B1 : Cfg::R_X2M + i1 + B1 * i3;
    const int r3p = (i3 + 1 < B3) ? rc + B1 * B2 : Cfg::R_X3P + i1 + B1 * i2;
    const int r3m = (i3 > 0) ? rc - B1 * B2 : Cfg::R_X3M + i1 + B1 * i2;
    uint32_t off[8];            // byte offsets of (neighbour site, component 0) inside a stage
    off[2] = r1p * Cfg::ROWB + h * 16;
    off[3] = r1m * Cfg::ROWB + h * 16;
    off[4] = r2p * Cfg::ROWB + h * 16;
    off[5] = r2m * Cfg::ROWB + h * 16;
    off[6] = r3p * Cfg::ROWB + h * 16;
    off[7] = r3m * Cfg::ROWB + h * 16;
    // byte offset of component k = spin*3 + C inside a row block [k][h] of 16-byte complex
    constexpr uint32_t KOFF0 = (0 * 3 + C) * LH * 16, KOFF1 = (1 * 3 + C) * LH * 16;
    constexpr uint32_t KOFF2 = (2 * 3 + C) * LH * 16, KOFF3 = (3 * 3 + C) * LH * 16;

    const long long nrow = (long long)args.L1 * args.L2 * args.L3;
    double2 *red = reinterpret_cast<double2 *>(smem + Cfg::NSTAGE * Cfg::STAGE_BYTES);
    double2 U[24];              // column C of the 8 links: U[leg*3 + a] = U_leg[a][C]

    int g = 0;
    for (int it = 0; it < my_tiles; it++) {
        const int4 o = args.tiles[blockIdx.x + it * gridDim.x];
        const int x1 = o.x + i1, x2 = o.y + i2, x3 = o.z + i3;
        const int r = (x1 + x2 + x3 + args.parity_out) & 1;          // x0 = 2h + r
        const long long grow = x1 + (long long)args.L1 * (x2 + (long long)args.L2 * x3);
        int hp = h + r;       if (hp == LH) hp = 0;
        int hm = h - 1 + r;   if (hm < 0) hm = LH - 1;
        off[0] = rc * Cfg::ROWB + hp * 16;
        off[1] = rc * Cfg::ROWB + hm * 16;
        {
            const double2 *gp = args.gauge + grow * (72 * LH) + 2 * h;
#pragma unroll
            for (int leg = 0; leg < 8; leg++)
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    const int f = leg * 9 + a * 3 + C;
                    U[leg * 3 + a] = __ldg(gp + (f >> 1) * 2 * LH + (f & 1));
                }
        }
        double2 *orow = args.out + grow * (12 * LH) + h;                // + s * nrow * 12 * LH + k * LH
        for (int s = 0; s < args.Ls; s++, g++) {
            const int stage = g & 1;
            // AXPY: this thread's four components of x, requested before the wait so that the global-memory
            // latency hides behind the legs
            double2 xv[4];
            if constexpr (AXPY) {
                if (active) {
                    const double2 *xp = args.axpy_x + (orow - args.out) + (long long)s * nrow * (12 * LH);
#pragma unroll
                    for (int j = 0; j < 4; j++) xv[j] = __ldcs(xp + (4 * C + j) * LH);
                }
            }
            mbar_wait(full_base + 8 * stage, (g >> 1) & 1);
            const unsigned char *sb = smem + stage * Cfg::STAGE_BYTES;
            double2 acc[12];
#pragma unroll
            for (int k = 0; k < 12; k++) acc[k] = make_double2(0.0, 0.0);
#define DWF_LEG64(L, MU, FWD)                                                                       \
            {                                                                                       \
                const unsigned char *nb = sb + off[L];                                              \
                leg64<MU, (FWD) != DAG>(acc, *reinterpret_cast<const double2 *>(nb + KOFF0),        \
                                        *reinterpret_cast<const double2 *>(nb + KOFF1),             \
                                        *reinterpret_cast<const double2 *>(nb + KOFF2),             \
                                        *reinterpret_cast<const double2 *>(nb + KOFF3), U + 3 * (L)); \
            }
            DWF_LEG64(0, 0, true)
            DWF_LEG64(1, 0, false)
            DWF_LEG64(2, 1, true)
            DWF_LEG64(3, 1, false)
            DWF_LEG64(4, 2, true)
            DWF_LEG64(5, 2, false)
            DWF_LEG64(6, 3, true)
            DWF_LEG64(7, 3, false)
#undef DWF_LEG64
            // this warp is done with the stage
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_base + 8 * stage);

            // exchange: thread C owns output components 4C .. 4C+3 and hands the other two blocks over
            const int buf = g & 1;
#pragma unroll
            for (int cc = 0; cc < 3; cc++) {
                if (cc == C) continue;
                const int slot = (C < cc) ? C : C - 1;
#pragma unroll
                for (int j = 0; j < 4; j++)
                    red[((((buf * 3 + cc) * 2 + slot) * 4 + j) * Cfg::TP) + site] = acc[4 * cc + j];
            }
            asm volatile("bar.sync %0, 96;" ::"r"(1 + (site >> 5)) : "memory");     // the three warps of this 32-site group
            if (active) {
                double2 *o2 = orow + (long long)s * nrow * (12 * LH);
#pragma unroll
                for (int j = 0; j < 4; j++) {
                    const double2 a0 = red[((((buf * 3 + C) * 2 + 0) * 4 + j) * Cfg::TP) + site];
                    const double2 a1 = red[((((buf * 3 + C) * 2 + 1) * 4 + j) * Cfg::TP) + site];
                    double2 v = cadd(cadd(acc[4 * C + j], a0), a1);
                    const int k = 4 * C + j;
                    if constexpr (AXPY) {
                        v.x = fma(args.axpy_b, v.x, args.axpy_a * xv[j].x);
                        v.y = fma(args.axpy_b, v.y, args.axpy_a * xv[j].y);
                    }
                    __stcs(o2 + k * LH, v);
                }
            }
        }
    }
}

template <int LH, int B1, int B2, int B3, bool DAG, bool AXPY>
__global__ void __launch_bounds__(Staged64Cfg<LH, B1, B2, B3>::NT, 1)
dhop_staged64_kernel(const __grid_constant__ CUtensorMap map_c, const __grid_constant__ CUtensorMap map_x1,
                     const __grid_constant__ CUtensorMap map_x2, const __grid_constant__ CUtensorMap map_x3,
                     const Staged64Args args)
{
    using Cfg = Staged64Cfg<LH, B1, B2, B3>;
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t full_base = smem_base + Cfg::NSTAGE * Cfg::STAGE_BYTES + Cfg::RED_BYTES;   // full[2]
    const uint32_t empty_base = full_base + 16;                                                // empty[2]
    const int tid = threadIdx.x;
    const int my_tiles = (args.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int nsteps = my_tiles * args.Ls;
    if (nsteps <= 0) return;
    if (tid == 0) {
        tma_prefetch_desc(&map_c);
        tma_prefetch_desc(&map_x1);
        tma_prefetch_desc(&map_x2);
        tma_prefetch_desc(&map_x3);
        for (int i = 0; i < 2; i++) {
            mbar_init(full_base + 8 * i, 1);
            mbar_init(empty_base + 8 * i, Cfg::NWARP_C);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (tid < 128) {            // producer warpgroup: one thread issues the seven boxes of every step
        reg_dealloc<Cfg::PROD_REGS>();
        if (tid != 0) return;
        const int L1 = args.L1, L2 = args.L2, L3 = args.L3;
        for (int g = 0; g < nsteps; g++) {
            const int it = g / args.Ls, s = g % args.Ls, stage = g & 1;
            if (g >= 2) mbar_wait(empty_base + 8 * stage, ((g >> 1) - 1) & 1);
            const int4 o = args.tiles[blockIdx.x + it * gridDim.x];
            const uint32_t bar = full_base + 8 * stage;
            const uint32_t dst = smem_base + stage * Cfg::STAGE_BYTES;
            const int sb = s * L3;                 // x3 and s share tensor dimension 4
            const int x1m = o.x == 0 ? L1 - 1 : o.x - 1, x1p = o.x + B1 == L1 ? 0 : o.x + B1;
            const int x2m = o.y == 0 ? L2 - 1 : o.y - 1, x2p = o.y + B2 == L2 ? 0 : o.y + B2;
            const int x3m = o.z == 0 ? L3 - 1 : o.z - 1, x3p = o.z + B3 == L3 ? 0 : o.z + B3;
            mbar_arrive_expect_tx(bar, Cfg::STAGE_BYTES);
            const int c4 = sb + o.z;
            tma_load_5d(dst, &map_c, bar, 0, 0, o.x, o.y, c4);
            tma_load_5d(dst + Cfg::R_X1M * Cfg::ROWB, &map_x1, bar, 0, 0, x1m, o.y, c4);
            tma_load_5d(dst + Cfg::R_X1P * Cfg::ROWB, &map_x1, bar, 0, 0, x1p, o.y, c4);
            tma_load_5d(dst + Cfg::R_X2M * Cfg::ROWB, &map_x2, bar, 0, 0, o.x, x2m, c4);
            tma_load_5d(dst + Cfg::R_X2P * Cfg::ROWB, &map_x2, bar, 0, 0, o.x, x2p, c4);
            tma_load_5d(dst + Cfg::R_X3M * Cfg::ROWB, &map_x3, bar, 0, 0, o.x, o.y, sb + x3m);
            tma_load_5d(dst + Cfg::R_X3P * Cfg::ROWB, &map_x3, bar, 0, 0, o.x, o.y, sb + x3p);
        }
        return;
    }

    reg_alloc<Cfg::CONS_REGS>();
    const int ctid = tid - 128;
    if (ctid >= 3 * Cfg::TP) return;
    const int c = ctid / Cfg::TP, site = ctid % Cfg::TP;         // colour-major: uniform per warp
    if (c == 0)      consume64<LH, B1, B2, B3, DAG, AXPY, 0>(args, smem, full_base, empty_base, site, my_tiles);
    else if (c == 1) consume64<LH, B1, B2, B3, DAG, AXPY, 1>(args, smem, full_base, empty_base, site, my_tiles);
    else             consume64<LH, B1, B2, B3, DAG, AXPY, 2>(args, smem, full_base, empty_base, site, my_tiles);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct Variant64 {
    int lh, b1, b2, b3, smem, threads;
    const void *fn[4];       // plain, dagger, a x + b Dhop, a x + b Dhop^dagger
};

#define DWF_STAGED64_VARIANTS(X) X(16, 2, 1, 2) X(16, 1, 1, 4) X(16, 1, 2, 2) X(16, 2, 2, 1) X(8, 4, 2, 1) X(8, 2, 2, 2) X(4, 4, 4, 1) X(4, 4, 2, 2) X(4, 2, 2, 2) X(4, 2, 2, 1) X(8, 2, 2, 1) X(16, 2, 1, 1)

static const std::vector<Variant64> &variants64()
{
    static const std::vector<Variant64> v = [] {
        std::vector<Variant64> t;
#define X(LH, B1, B2, B3)                                                                             \
        t.push_back({LH, B1, B2, B3, Staged64Cfg<LH, B1, B2, B3>::SMEM_BYTES, Staged64Cfg<LH, B1, B2, B3>::NT, \
                     {reinterpret_cast<const void *>(&dhop_staged64_kernel<LH, B1, B2, B3, false, false>),    \
                      reinterpret_cast<const void *>(&dhop_staged64_kernel<LH, B1, B2, B3, true, false>),     \
                      reinterpret_cast<const void *>(&dhop_staged64_kernel<LH, B1, B2, B3, false, true>),     \
                      reinterpret_cast<const void *>(&dhop_staged64_kernel<LH, B1, B2, B3, true, true>)}});
        DWF_STAGED64_VARIANTS(X)
#undef X
        return t;
    }();
    return v;
}

void plan_staged64(dwf_geometry *g)
{
    g->staged64.variant = -1;
    if (g->prec != DWF_F64 || !get_tensor_map_encoder()) return;
    const Lattice &lat = g->lat;
    const std::vector<Variant64> &v = variants64();
    for (size_t i = 0; i < v.size(); i++) {
        if (v[i].lh != lat.Lh) continue;
        if (lat.L[1] % v[i].b1 || lat.L[2] % v[i].b2 || lat.L[3] % v[i].b3) continue;
        if (g->opt_variant > 0 && (int)i + 1 != g->opt_variant) continue;
        g->staged64.variant = (int)i;
        g->staged64.b[0] = v[i].b1; g->staged64.b[1] = v[i].b2; g->staged64.b[2] = v[i].b3;
        g->staged64.ntiles = (lat.L[1] / v[i].b1) * (lat.L[2] / v[i].b2) * (lat.L[3] / v[i].b3);
        // per-device opt-in to the large dynamic shared memory (the caller holds a DeviceGuard)
        for (int d = 0; d < 4; d++)
            if (cudaFuncSetAttribute(v[i].fn[d], cudaFuncAttributeMaxDynamicSharedMemorySize, v[i].smem) != cudaSuccess) {
                cudaGetLastError();
                g->staged64.variant = -1;
            }
        return;
    }
}

// launch order of the row boxes: x1 fastest, x3 slowest, direction 2 split into macro blocks of at most
// 96 tile columns per x3 layer that are swept one after the other (as in dhop_staged.cu: the CTAs
// resident at one time then cover several x3 layers of a macro block and share their faces in L2)
void build_staged64_tile_table(const dwf_geometry *g, int4 *tab)
{
    const Lattice &lat = g->lat;
    const int *b = g->staged64.b;
    const int n1 = lat.L[1] / b[0], n2 = lat.L[2] / b[1], n3 = lat.L[3] / b[2];
    int nsplit = 1;
    if (g->opt_raster_staged < 0) {
        while (n1 * (n2 / nsplit) > 96 && n2 % (nsplit * 2) == 0) nsplit *= 2;
    } else {
        for (int i = 0; i < g->opt_raster_staged % 10 && n2 % (nsplit * 2) == 0; i++) nsplit *= 2;
    }
    const int n2in = n2 / nsplit;
    int id = 0;
    for (int m = 0; m < nsplit; m++)
        for (int t3 = 0; t3 < n3; t3++)
            for (int t2 = 0; t2 < n2in; t2++)
                for (int t1 = 0; t1 < n1; t1++)
                    tab[id++] = make_int4(t1 * b[0], (m * n2in + t2) * b[1], t3 * b[2], 0);
}

// tensor map of an fp64 half field complex[s][x3][x2][x1][k][h] seen as 5-D fp64 tensor
// (2*Lh, 12, L1, L2, L3*Ls)
static int encode_map64(CUtensorMap *m, const void *base, const Lattice &lat, int b1, int b2, int b3)
{
    PFN_tensorMapEncodeTiled enc = get_tensor_map_encoder();
    const cuuint64_t dims[5] = {(cuuint64_t)2 * lat.Lh, 12, (cuuint64_t)lat.L[1], (cuuint64_t)lat.L[2],
                                (cuuint64_t)lat.L[3] * lat.Ls};
    const cuuint64_t krow = (cuuint64_t)lat.Lh * 16, row = 12 * krow;
    const cuuint64_t strides[4] = {krow, row, row * lat.L[1], row * lat.L[1] * lat.L[2]};
    const cuuint32_t box[5] = {(cuuint32_t)2 * lat.Lh, 12, (cuuint32_t)b1, (cuuint32_t)b2, (cuuint32_t)b3};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult rc = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<void *>(base), dims, strides, box, estr,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) {
        set_error("cuTensorMapEncodeTiled (fp64) failed with code %d", (int)rc);
        return DWF_ERR_CUDA;
    }
    return DWF_OK;
}

int launch_dhop_staged64(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st, bool dagger,
                         const void *axpy_x, double axpy_a, double axpy_b)
{
    const Variant64 &v = variants64()[(size_t)g->staged64.variant];
    CUtensorMap mc, m1, m2, m3;
    int rc;
    if ((rc = encode_map64(&mc, in, g->lat, v.b1, v.b2, v.b3))) return rc;
    if ((rc = encode_map64(&m1, in, g->lat, 1, v.b2, v.b3))) return rc;
    if ((rc = encode_map64(&m2, in, g->lat, v.b1, 1, v.b3))) return rc;
    if ((rc = encode_map64(&m3, in, g->lat, v.b1, v.b2, 1))) return rc;
    Staged64Args a;
    a.out = static_cast<double2 *>(out);
    a.gauge = static_cast<const double2 *>(g->gauge[parity_out]);
    a.tiles = g->tiles_staged64;
    a.ntiles = g->staged64.ntiles;
    a.L1 = g->lat.L[1]; a.L2 = g->lat.L[2]; a.L3 = g->lat.L[3]; a.Ls = g->lat.Ls;
    a.parity_out = parity_out;
    a.axpy_x = static_cast<const double2 *>(axpy_x);
    a.axpy_a = axpy_a;
    a.axpy_b = axpy_b;
    const void *fn = v.fn[(dagger ? 1 : 0) + (axpy_x ? 2 : 0)];
    const int grid = g->staged64.ntiles < g->sm_count ? g->staged64.ntiles : g->sm_count;
    void *params[] = {&mc, &m1, &m2, &m3, &a};
    DWF_CUDA_CHECK(cudaLaunchKernel(fn, dim3((unsigned)grid), dim3((unsigned)v.threads), params, (size_t)v.smem, st));
    count_launch();
    return DWF_OK;
}

}  // namespace dwf

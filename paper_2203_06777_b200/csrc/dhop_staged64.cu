// dhop_staged64.cu -- the fp64 TMA-staged Dhop kernels for sm_100a.  Three kernels, in the order of preference of
// the host tables: the site-per-thread kernel with the links in tensor memory (dhop_staged64s_kernel, second half of
// this file; 128-site tiles), and the two colour-split kernels described first: links of a site split by COLOUR COLUMN
// over three threads, kept in tensor memory (128-site tiles) or in registers (64-site tiles, every row length).
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
// store.  The exchange is deferred by one step and signalled through mbarriers (consume64), so no warp
// waits for its partners inside a step.  Threads are colour-major (a warp = one colour of 32 consecutive
// sites), so every LDS / STG is conflict-free and coalesced and there is no divergence.
// Everything else follows dhop_staged.cu: a producer warpgroup (setmaxnreg) issues 5-D bulk tensor
// copies (TMA) of the input slice -- rows box + 6 faces -- into a two-stage shared-memory ring with
// full / empty mbarriers; consumers walk all Ls slices of a tile with their link columns in registers.
// TMEM variant (template flag TM, tiles of 128 sites, preferred when the lattice fits): the link columns and the
// exchanged partial sums live in tensor memory (tcgen05.alloc / st / ld, shape 32x32b, as thread-private storage:
// "tensor memory as thread-private storage" below), which frees 96 registers and the shared-memory exchange buffer:
// twelve consumer warps instead of six and a 4x instead of 5x halo.
// Layouts (pack.cu): spinor complex[s][row][k][h], k = spin*3 + colour (one plane per component:
// consecutive sites are consecutive 128-bit words); links
// complex[row][f/2][h][f&1], f = leg*9 + a*3 + b.
#include <type_traits>
#include <vector>

#include "complex_ops.cuh"
#include "dwf_internal.cuh"
#include "tma.cuh"

namespace dwf {

#ifndef DWF_STAGED64_MODE
#define DWF_STAGED64_MODE 0     // which kernel MODE this translation unit instantiates (build.py compiles the file once per MODE)
#endif

PFN_tensorMapEncodeTiled get_tensor_map_encoder();      // dhop_staged.cu

struct Staged64Args {
    double2 *out;
    const double2 *gauge;    // gauge set of the output parity: [row][36 pairs][Lh][2]
    const int4 *tiles;       // origins (o1, o2, o3) of the row boxes, launch order
    int ntiles;
    int L1, L2, L3, Ls;
    int parity_out;
    int zigzag;              // walk the slices of every other tile backwards (L2 reuse between tiles)
    int l2pol;               // decimal digits: digit 0 input boxes, 6 links, 7 output (0 normal, 1 evict_first, 2 evict_last)
    uint32_t zero;           // 0 at run time, unknown to ptxas: makes the release of a stage depend on the loaded data (tma.cuh)
    const double2 *axpy_x;   // AXPY kernels: out = a x + b Dhop in (x on the output parity; may be out)
    double axpy_a, axpy_b;
    double *norm_partials;   // NORM kernels: one partial sum of |out|^2 per CTA (fixed order inside the CTA)
};

// TM: the TMEM variant (tiles of 128 sites): link columns and the colour exchange live in tensor memory
template <int LH, int B1, int B2, int B3, bool TM = false> struct Staged64Cfg {
    static constexpr int NROW_C = B1 * B2 * B3;
    static constexpr int T = LH * NROW_C;                        // output sites per tile
    static constexpr int TP = (T + 31) / 32 * 32;                // sites padded to whole warps: thread = colour * TP + site
    static constexpr int NGROUP = TP / 32;                       // 32-site groups: three warps (one per colour) each
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
    static constexpr int RED_BYTES = TM ? 0 : 2 * 3 * 2 * 4 * TP * 16;
    // tail: full[2], empty[2][4 regions], exch[NGROUP][2] mbarriers, one fp64 slot per consumer warp (fused norm2)
    static constexpr int TAIL_EXCH = 16 + 64, TAIL_NORM = TAIL_EXCH + 16 * NGROUP, TAIL_TMEM = TAIL_NORM + 8 * NWARP_C, TAIL = TAIL_TMEM + 8;
    static constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + RED_BYTES + (TAIL + 15) / 16 * 16;
    static constexpr int PROD_REGS = 24;
    static constexpr int CONS_REGS_RAW = ((65536 - 128 * PROD_REGS) / NTC) / 8 * 8;
    static constexpr int CONS_REGS = CONS_REGS_RAW > 240 ? 240 : CONS_REGS_RAW;
    static_assert(ROWB % 128 == 0, "staged rows must keep TMA destinations 128-byte aligned");
    static_assert(SMEM_BYTES <= 232448, "tile too large for shared memory");
    static_assert(!TM || NGROUP == 4, "the TMEM variant needs 128-site tiles: the three colour warps of a site group must share a lane quadrant");
};

__device__ __forceinline__ double2 ldg_d2_hint(const double2 *p, uint64_t policy)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(policy));
    return v;
}
// two consecutive complex numbers (32 bytes, 32-byte aligned) in one 256-bit load
__device__ __forceinline__ void ldg_d4_hint(const double2 *p, uint64_t policy, double2 &a, double2 &b)
{
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f64 {%0, %1, %2, %3}, [%4], %5;"
                 : "=d"(a.x), "=d"(a.y), "=d"(b.x), "=d"(b.y) : "l"(p), "l"(policy));
}
__device__ __forceinline__ void stg_d2_hint(double2 *p, double2 v, uint64_t policy)
{
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(policy) : "memory");
}

// ---- tensor memory (TMEM) as thread-private storage -------------------------------------------------
// tcgen05.ld / tcgen05.st with shape 32x32b: lane i of a warp reads / writes N consecutive 32-bit columns of TMEM
// lane (32 * (warp % 4) + i).  Consumer warp w = colour * 4 + group sits in lane quadrant group (the CTA's first
// four warps are the producer warpgroup), so the three colour threads of a site share ONE TMEM lane:
//   columns [96 c, 96 c + 96)                        the link column of colour c: leg L at +12 L (3 complex = 12 words)
//   columns [288 + 96 b + 32 c, +32), b = 0, 1       exchange buffer b written by colour c: block r = 1 at +0, r = 2 at +16
// 480 of the 512 columns.  Measured (profiles/r02_tmem_microbench.md): >= 314 B/clk/SM with 12 warps, 2.5 x shared memory.
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr));
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t (&r)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
// the 12 words of one leg's link column: columns [taddr, taddr + 12) as an x8 and an x4 load
__device__ __forceinline__ void tmem_ld12(uint32_t taddr, uint32_t (&r)[3][4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0][0]), "=r"(r[0][1]), "=r"(r[0][2]), "=r"(r[0][3]), "=r"(r[1][0]), "=r"(r[1][1]), "=r"(r[1][2]), "=r"(r[1][3]) : "r"(taddr));
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r[2][0]), "=r"(r[2][1]), "=r"(r[2][2]), "=r"(r[2][3]) : "r"(taddr + 8));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                   "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]) : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
                   "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]),
                   "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
}
__device__ __forceinline__ void tmem_pack(uint32_t *r, double2 v)
{
    r[0] = (uint32_t)__double2loint(v.x); r[1] = (uint32_t)__double2hiint(v.x);
    r[2] = (uint32_t)__double2loint(v.y); r[3] = (uint32_t)__double2hiint(v.y);
}
__device__ __forceinline__ double2 tmem_unpack_p(const uint32_t *r)
{
    return make_double2(__hiloint2double((int)r[1], (int)r[0]), __hiloint2double((int)r[3], (int)r[2]));
}
// one complex fp64 number = four columns
__device__ __forceinline__ void tmem_st_c(uint32_t taddr, double2 v)
{
    uint32_t r[4] = {(uint32_t)__double2loint(v.x), (uint32_t)__double2hiint(v.x), (uint32_t)__double2loint(v.y), (uint32_t)__double2hiint(v.y)};
    tmem_st4(taddr, r);
}
__device__ __forceinline__ double2 tmem_unpack(const uint32_t (&r)[4])
{
    return make_double2(__hiloint2double((int)r[1], (int)r[0]), __hiloint2double((int)r[3], (int)r[2]));
}
// tcgen05.ld is asynchronous: its destination registers are valid only after tcgen05.wait::ld.  The registers are
// in/out operands of the wait, so that every later use depends on it -- without a memory clobber, which would keep
// ptxas from moving the shared-memory loads of the next legs across it.
__device__ __forceinline__ void tmem_wait_ld_regs3(uint32_t (&w)[3][4])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(w[0][0]), "+r"(w[0][1]), "+r"(w[0][2]), "+r"(w[0][3]), "+r"(w[1][0]), "+r"(w[1][1]), "+r"(w[1][2]), "+r"(w[1][3]),
                   "+r"(w[2][0]), "+r"(w[2][1]), "+r"(w[2][2]), "+r"(w[2][3]));
}
__device__ __forceinline__ void tmem_wait_ld_regs(uint32_t (&a)[16], uint32_t (&b)[16])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]), "+r"(a[7]), "+r"(a[8]), "+r"(a[9]), "+r"(a[10]),
                   "+r"(a[11]), "+r"(a[12]), "+r"(a[13]), "+r"(a[14]), "+r"(a[15]), "+r"(b[0]), "+r"(b[1]), "+r"(b[2]), "+r"(b[3]), "+r"(b[4]), "+r"(b[5]),
                   "+r"(b[6]), "+r"(b[7]), "+r"(b[8]), "+r"(b[9]), "+r"(b[10]), "+r"(b[11]), "+r"(b[12]), "+r"(b[13]), "+r"(b[14]), "+r"(b[15]));
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// one leg for colour column c: acc += reconstruct( U[:, c] * project(psi)[c] ).  p0..p3 = colour c of the
// four spin components of the neighbour; U[r] = U_{(c+r)%3, c}, r = 0..2 (the rows of the column ROTATED
// by the thread's colour, so that acc[spin*3 + r] is the partial sum for output colour (c+r)%3 and every
// register index is a compile-time constant although c is a run-time value: one copy of the code for all
// three colours).  Signs as in dhop.cu (DeGrand-Rossi).  FIRST: the leg that initialises the accumulators.
template <int MU, bool FWD, bool FIRST>
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
        if constexpr (FIRST) {
            acc[0 + a] = x0;
            acc[3 + a] = x1;
            if constexpr (MU == 0) {
                acc[6 + a] = FWD ? cmuli(x1) : cmulni(x1);
                acc[9 + a] = FWD ? cmuli(x0) : cmulni(x0);
            } else if constexpr (MU == 1) {
                acc[6 + a] = FWD ? cneg(x1) : x1;
                acc[9 + a] = FWD ? x0 : cneg(x0);
            } else if constexpr (MU == 2) {
                acc[6 + a] = FWD ? cmuli(x0) : cmulni(x0);
                acc[9 + a] = FWD ? cmulni(x1) : cmuli(x1);
            } else {
                acc[6 + a] = FWD ? cneg(x0) : x0;
                acc[9 + a] = FWD ? cneg(x1) : x1;
            }
        } else {
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
}

// MODE bits: 1 = Dhop^dagger (projectors swapped), 2 = a x + b Dhop in the store epilogue, 4 = |out|^2
// accumulated in the store epilogue (fused norm2; not combined with the others).
//
// Consumer body of thread (site, colour c); c is uniform in a warp.  Thread c ends up owning output colour
// c (four spin components): of its 12 partial sums acc[spin*3 + r] it keeps the block r = 0 and hands the
// blocks r = 1, 2 to the threads of colours (c+1)%3, (c+2)%3 through shared memory.
// The colour exchange is DEFERRED by one step: after the 8 legs of step g a warp first finishes step g-1
// (waits on that step's exchange mbarrier -- long since complete --, adds the two partial sums of its
// partner warps to the block it kept in registers, stores), then publishes its own partial sums of step g
// and arrives on the mbarrier of step g.  No warp waits for its partners inside a step; the three colour
// warps of a 32-site group drift by up to one step.  Two exchange buffers suffice: a buffer is overwritten
// at step g+2, after this warp has seen all arrivals of step g+1, each of which follows that warp's reads
// of step g.
template <int LH, int B1, int B2, int B3, int MODE, bool TM>
__device__ __forceinline__ void consume64(const Staged64Args &args, unsigned char *smem, const uint32_t full_base,
                                          const uint32_t empty_base, const uint32_t exch_base, const int site, const int c,
                                          const int my_tiles, double &nsum, const uint32_t tmem_base)
{
    using Cfg = Staged64Cfg<LH, B1, B2, B3, TM>;
    constexpr bool DAG = (MODE & 1) != 0, AXPY = (MODE & 2) != 0, NORM = (MODE & 4) != 0;
    const bool active = site < Cfg::T;
    const int st = active ? site : 0;
    const int h = st % LH, row = st / LH;
    const int i1 = row % B1, i2 = (row / B1) % B2, i3 = row / (B1 * B2);
    const int lane = threadIdx.x & 31;
    // L2 eviction classes of the global accesses: option "l2pol", digits as in dhop_staged.cu (PC_*)
    const uint64_t pol_first = l2_policy(args.l2pol / 1000000 % 10), pol_out = l2_policy(args.l2pol / 10000000 % 10);

    // staged rows of the 8 neighbours (tile-invariant except the x0 pair)
    const int rc = row;
    const int r1p = (i1 + 1 < B1) ? rc + 1 : Cfg::R_X1P + i2 + B2 * i3;
    const int r1m = (i1 > 0) ? rc - 1 : Cfg::R_X1M + i2 + B2 * i3;
    const int r2p = (i2 + 1 < B2) ? rc + B1 : Cfg::R_X2P + i1 + B1 * i3;
    const int r2m = (i2 > 0) ? rc - B1 : Cfg::R_X2M + i1 + B1 * i3;
    const int r3p = (i3 + 1 < B3) ? rc + B1 * B2 : Cfg::R_X3P + i1 + B1 * i2;
    const int r3m = (i3 > 0) ? rc - B1 * B2 : Cfg::R_X3M + i1 + B1 * i2;
    // byte offsets of (neighbour site, component k = 0*3 + c) inside a stage; the other three spin
    // components of colour c follow at multiples of KSPIN
    const uint32_t coff = (uint32_t)(c * LH + h) * 16;
    constexpr uint32_t KSPIN = 3 * LH * 16;
    uint32_t off[8];
    off[2] = r1p * Cfg::ROWB + coff;
    off[3] = r1m * Cfg::ROWB + coff;
    off[4] = r2p * Cfg::ROWB + coff;
    off[5] = r2m * Cfg::ROWB + coff;
    off[6] = r3p * Cfg::ROWB + coff;
    off[7] = r3m * Cfg::ROWB + coff;

    const long long nrow = (long long)args.L1 * args.L2 * args.L3;
    // exchange buffer [buf][destination colour d][slot][spin j][site]: slot 0 comes from colour (d+2)%3
    // (its block r = 1), slot 1 from colour (d+1)%3 (its block r = 2)
    double2 *red = reinterpret_cast<double2 *>(smem + Cfg::NSTAGE * Cfg::STAGE_BYTES);
    const int c1 = c == 2 ? 0 : c + 1, c2 = c == 0 ? 2 : c - 1;        // (c+1)%3, (c+2)%3
    double2 *red_w1 = red + (size_t)((c1 * 2 + 0) * 4) * Cfg::TP + site;   // my block r = 1 -> colour c1, slot 0
    double2 *red_w2 = red + (size_t)((c2 * 2 + 1) * 4) * Cfg::TP + site;   // my block r = 2 -> colour c2, slot 1
    const double2 *red_r = red + (size_t)((c * 2) * 4) * Cfg::TP + site;   // what the partners left for colour c
    constexpr int RED_BUF = 3 * 2 * 4 * Cfg::TP;                            // complex numbers per buffer
    const uint32_t my_exch = exch_base + 16 * (site >> 5);      // exch[group][2]
    // column c of the 8 links, rows rotated: U[leg*3 + r] = U_leg[(c+r)%3][c]; in registers, or (TM) in tensor memory
    double2 U[TM ? 1 : 24];
    // TM: this thread's TMEM lane is 32 * group + lane (group = site >> 5 = warp % 4); column ranges as above
    const uint32_t tm_lane = tmem_base + ((uint32_t)((site >> 5) * 32) << 16);
    const uint32_t tm_links = tm_lane + 96u * c;
    const uint32_t tm_xw = tm_lane + 288u + 32u * c;                                   // where I publish (+ 96 buf)
    const uint32_t tm_xr0 = tm_lane + 288u + 32u * c2, tm_xr1 = tm_lane + 288u + 32u * c1 + 16u;   // what is left for me

    // global row of this thread's site in the it-th tile, and the parity bit r of x0 = 2h + r
    auto tile_row = [&](int it, int &r) -> long long {
        const int4 o = args.tiles[blockIdx.x + it * gridDim.x];
        const int x1 = o.x + i1, x2 = o.y + i2, x3 = o.z + i3;
        r = (x1 + x2 + x3 + args.parity_out) & 1;
        return x1 + (long long)args.L1 * (x2 + (long long)args.L2 * x3);
    };
    auto set_x0_offsets = [&](int r) {
        int hp = h + r;       if (hp == LH) hp = 0;
        int hm = h - 1 + r;   if (hm < 0) hm = LH - 1;
        off[0] = rc * Cfg::ROWB + (uint32_t)(c * LH + hp) * 16;
        off[1] = rc * Cfg::ROWB + (uint32_t)(c * LH + hm) * 16;
    };
    const int rot[3] = {c, c1, c2};
    auto load_links = [&](long long grow) {
        const double2 *gp = args.gauge + grow * (72 * LH) + 2 * h;
        if constexpr (TM) {
            double2 t[24];
#pragma unroll
            for (int leg = 0; leg < 8; leg++)
#pragma unroll
                for (int r = 0; r < 3; r++) {
                    const int f = leg * 9 + rot[r] * 3 + c;
                    t[leg * 3 + r] = ldg_d2_hint(gp + (f >> 1) * 2 * LH + (f & 1), pol_first);
                }
#pragma unroll
            for (int k = 0; k < 24; k++) tmem_st_c(tm_links + 4 * k, t[k]);
            tmem_wait_st();
        } else {
#pragma unroll
            for (int leg = 0; leg < 8; leg++)
#pragma unroll
                for (int r = 0; r < 3; r++) {
                    const int f = leg * 9 + rot[r] * 3 + c;
                    U[leg * 3 + r] = ldg_d2_hint(gp + (f >> 1) * 2 * LH + (f & 1), pol_first);
                }
        }
    };

    // the pending step: the block of partial sums this thread owns, where it goes, its x (AXPY)
    double2 keep[4], xk[4];
    double2 *keep_o = nullptr;
    int keep_g = -1;
    auto finish = [&]() {
        const int buf = keep_g & 1;
        mbar_wait(my_exch + 8 * buf, (keep_g >> 1) & 1);
        if (active) {
            double2 a0[4], a1[4];
            if constexpr (TM) {
                tmem_fence_after();
                uint32_t w0[16], w1[16];
                tmem_ld16(tm_xr0 + 96u * buf, w0);
                tmem_ld16(tm_xr1 + 96u * buf, w1);
                tmem_wait_ld_regs(w0, w1);
#pragma unroll
                for (int j = 0; j < 4; j++) { a0[j] = tmem_unpack_p(w0 + 4 * j); a1[j] = tmem_unpack_p(w1 + 4 * j); }
            } else {
#pragma unroll
                for (int j = 0; j < 4; j++) {
                    a0[j] = red_r[buf * RED_BUF + j * Cfg::TP];
                    a1[j] = red_r[buf * RED_BUF + (4 + j) * Cfg::TP];
                }
            }
            double2 v[4];
#pragma unroll
            for (int j = 0; j < 4; j++) {
                v[j] = cadd(cadd(keep[j], a0[j]), a1[j]);
                if constexpr (AXPY) {
                    v[j].x = fma(args.axpy_b, v[j].x, args.axpy_a * xk[j].x);
                    v[j].y = fma(args.axpy_b, v[j].y, args.axpy_a * xk[j].y);
                }
                if constexpr (NORM) nsum = fma(v[j].x, v[j].x, fma(v[j].y, v[j].y, nsum));
            }
#pragma unroll
            for (int j = 0; j < 4; j++) stg_d2_hint(keep_o + (3 * j) * LH, v[j], pol_out);      // component k = j*3 + c
        }
    };

    int r_cur;
    long long grow = tile_row(0, r_cur);
    set_x0_offsets(r_cur);
    load_links(grow);

    // One slice: 8 legs out of the staged buffer, then the deferred finish of the previous slice
    auto step = [&](const int g, const int s) {
        const int stage = g & 1;
        const uint32_t eb = empty_base + 32 * stage;
        double2 *o2 = args.out + grow * (12 * LH) + (c * LH + h) + (long long)s * nrow * (12 * LH);
        // AXPY: this thread's four components of x, requested before the wait so that the global-memory
        // latency hides behind the legs
        double2 xv[4];
        if constexpr (AXPY) {
            if (active) {
                const double2 *xp = args.axpy_x + (o2 - args.out);
#pragma unroll
                for (int j = 0; j < 4; j++) xv[j] = __ldcs(xp + (3 * j) * LH);
            }
        }
        mbar_wait(full_base + 8 * stage, (g >> 1) & 1);
        const unsigned char *sb = smem + stage * Cfg::STAGE_BYTES;
        double2 acc[12];
        // the four loads of leg L (colour c of the four spin components of the neighbour), then the leg
#define DWF_LOAD64(L)                                                                               \
        const double2 q##L##_0 = *reinterpret_cast<const double2 *>(sb + off[L]),                    \
                      q##L##_1 = *reinterpret_cast<const double2 *>(sb + off[L] + KSPIN),            \
                      q##L##_2 = *reinterpret_cast<const double2 *>(sb + off[L] + 2 * KSPIN),        \
                      q##L##_3 = *reinterpret_cast<const double2 *>(sb + off[L] + 3 * KSPIN);
        // TM: the three link elements of leg L come out of tensor memory, requested two legs ahead: tcgen05.wait::ld
        // waits for ALL loads in flight, so the request for leg NEXT goes out right after the wait of leg L, into the
        // registers leg L has just been unpacked from, and lands during the arithmetic of leg L.
#define DWF_TLOAD(L, W)                                                                             \
        if constexpr (TM) { tmem_ld12(tm_links + 12 * (L), W); }
#define DWF_LEG64(L, MU, FWD, FIRST, W, NEXT)                                                       \
        if constexpr (TM) {                                                                         \
            tmem_wait_ld_regs3(W);                                                                  \
            const double2 Ul[3] = {tmem_unpack(W[0]), tmem_unpack(W[1]), tmem_unpack(W[2])};        \
            if constexpr ((NEXT) >= 0) { DWF_TLOAD((NEXT) < 0 ? 0 : (NEXT), W) }                    \
            leg64<MU, (FWD) != DAG, FIRST>(acc, q##L##_0, q##L##_1, q##L##_2, q##L##_3, Ul);        \
        } else {                                                                                    \
            leg64<MU, (FWD) != DAG, FIRST>(acc, q##L##_0, q##L##_1, q##L##_2, q##L##_3, U + 3 * (L)); \
        }
        // Legs in the order x3, x2, x1, x0.  The stage is handed back to the producer ONCE, after the last leg: warp
        // barrier, then lane 0's four arrives, whose addresses are computed from acc[0].x and acc[3].x (spin components 0
        // and 1 of the rotated colour 0: together they derive from all four loads of every leg), so that no arrive can issue
        // while a load of the stage is in flight (tma.cuh: mbar_arrive_dep).  Releasing the face regions right after the two
        // legs that read them (as dhop_staged.cu does) is correct with the same kind of arrive but not faster here (1033 vs
        // 1025 us), so it is not used.
        uint32_t ua[3][4], ub[3][4];
        DWF_TLOAD(6, ua)
        DWF_TLOAD(7, ub)
        DWF_LOAD64(6) DWF_LOAD64(7)
        DWF_LEG64(6, 3, true, true, ua, 4)
        DWF_LEG64(7, 3, false, false, ub, 5)
        DWF_LOAD64(4) DWF_LOAD64(5)
        DWF_LEG64(4, 2, true, false, ua, 2)
        DWF_LEG64(5, 2, false, false, ub, 3)
        DWF_LOAD64(2) DWF_LOAD64(3)
        DWF_LEG64(2, 1, true, false, ua, 0)
        DWF_LEG64(3, 1, false, false, ub, 1)
        DWF_LOAD64(0) DWF_LOAD64(1)
        DWF_LEG64(0, 0, true, false, ua, -1)
        DWF_LEG64(1, 0, false, false, ub, -1)
        __syncwarp();
        if (lane == 0) {
            mbar_arrive_dep(eb, args.zero, acc[0].x, acc[3].x);
            mbar_arrive_dep(eb + 8, args.zero, acc[0].x, acc[3].x);
            mbar_arrive_dep(eb + 16, args.zero, acc[0].x, acc[3].x);
            mbar_arrive_dep(eb + 24, args.zero, acc[0].x, acc[3].x);
        }
#undef DWF_LOAD64
#undef DWF_LEG64
#undef DWF_TLOAD

        if (keep_g >= 0) finish();               // the previous step: its exchange has long completed
        // publish the blocks r = 1, 2 of this step
        const int buf = g & 1;
        if constexpr (TM) {
            uint32_t w[32];
#pragma unroll
            for (int j = 0; j < 4; j++) {
                tmem_pack(w + 4 * j, acc[3 * j + 1]);
                tmem_pack(w + 16 + 4 * j, acc[3 * j + 2]);
            }
            tmem_st32(tm_xw + 96u * buf, w);
            tmem_wait_st();
            tmem_fence_before();
        } else {
#pragma unroll
            for (int j = 0; j < 4; j++) {
                red_w1[buf * RED_BUF + j * Cfg::TP] = acc[3 * j + 1];
                red_w2[buf * RED_BUF + j * Cfg::TP] = acc[3 * j + 2];
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(my_exch + 8 * buf);
#pragma unroll
        for (int j = 0; j < 4; j++) {
            keep[j] = acc[3 * j];
            if constexpr (AXPY) xk[j] = xv[j];
        }
        keep_o = o2;
        keep_g = g;
    };

    int g = 0;
    for (int it = 0; it < my_tiles; it++) {
        const bool has_next = it + 1 < my_tiles;
        int r_next = r_cur;
        long long grow_next = grow;
        if (has_next) grow_next = tile_row(it + 1, r_next);
        for (int s = 0; s < args.Ls; s++, g++) {
            const int sl = (args.zigzag && (it & 1)) ? args.Ls - 1 - s : s;
            step(g, sl);
        }
        grow = grow_next;
        r_cur = r_next;
        set_x0_offsets(r_cur);
        // links of the next tile (a second code copy that refills them leg by leg during the last slice, as
        // dhop_staged.cu does, measured slower here: 1493 vs 1306 us on C4 -- instruction-cache misses)
        if (has_next) load_links(grow);
    }
    if (keep_g >= 0) finish();
}

template <int LH, int B1, int B2, int B3, int MODE, bool TM>
__global__ void __launch_bounds__(Staged64Cfg<LH, B1, B2, B3, TM>::NT, 1)
dhop_staged64_kernel(const __grid_constant__ CUtensorMap map_c, const __grid_constant__ CUtensorMap map_x1,
                     const __grid_constant__ CUtensorMap map_x2, const __grid_constant__ CUtensorMap map_x3,
                     const Staged64Args args)
{
    using Cfg = Staged64Cfg<LH, B1, B2, B3, TM>;
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t full_base = smem_base + Cfg::NSTAGE * Cfg::STAGE_BYTES + Cfg::RED_BYTES;   // full[2]
    const uint32_t empty_base = full_base + 16;                                                // empty[2][4 regions]
    const uint32_t exch_base = full_base + Cfg::TAIL_EXCH;                                     // exch[NGROUP][2]
    const int tid = threadIdx.x;
    const int my_tiles = (args.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int nsteps = my_tiles * args.Ls;
    if (nsteps <= 0) {
        if ((MODE & 4) && tid == 0) args.norm_partials[blockIdx.x] = 0.0;
        return;
    }
    if (tid == 0) {
        tma_prefetch_desc(&map_c);
        tma_prefetch_desc(&map_x1);
        tma_prefetch_desc(&map_x2);
        tma_prefetch_desc(&map_x3);
        for (int i = 0; i < 2; i++) mbar_init(full_base + 8 * i, 4);        // four regions arrive (expect_tx) per stage
        for (int i = 0; i < 8; i++) mbar_init(empty_base + 8 * i, Cfg::NWARP_C);
        for (int i = 0; i < 2 * Cfg::NGROUP; i++) mbar_init(exch_base + 8 * i, 3);
        mbar_fence_init();
    }
    // TM: warp 0 allocates all 512 columns of tensor memory (one CTA per SM) and leaves the base address in shared memory
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + Cfg::NSTAGE * Cfg::STAGE_BYTES + Cfg::RED_BYTES + Cfg::TAIL_TMEM);
    if constexpr (TM) {
        if (tid < 32) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(512) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        tmem_fence_before();
    }
    __syncthreads();
    uint32_t tmem_base = 0;
    if constexpr (TM) {
        tmem_fence_after();
        tmem_base = *tmem_slot;
    }

    if (tid < 128) {            // producer warpgroup: one thread issues the seven boxes of every step
        reg_dealloc<Cfg::PROD_REGS>();
        if (TM ? tid >= 32 : tid != 0) return;
        if (tid == 0) {
        const int L1 = args.L1, L2 = args.L2, L3 = args.L3;
        const uint64_t pol_last = l2_policy(args.l2pol % 10);      // input boxes are re-read by neighbouring tiles
        for (int g = 0; g < nsteps; g++) {
            const int it = g / args.Ls, i = g % args.Ls, stage = g & 1;
            const int s = (args.zigzag && (it & 1)) ? args.Ls - 1 - i : i;
            const int4 o = args.tiles[blockIdx.x + it * gridDim.x];
            const uint32_t bar = full_base + 8 * stage, eb = empty_base + 32 * stage;
            const uint32_t epar = ((g >> 1) - 1) & 1;
            const uint32_t dst = smem_base + stage * Cfg::STAGE_BYTES;
            const int sb = s * L3;                 // x3 and s share tensor dimension 4
            const int x1m = o.x == 0 ? L1 - 1 : o.x - 1, x1p = o.x + B1 == L1 ? 0 : o.x + B1;
            const int x2m = o.y == 0 ? L2 - 1 : o.y - 1, x2p = o.y + B2 == L2 ? 0 : o.y + B2;
            const int x3m = o.z == 0 ? L3 - 1 : o.z - 1, x3p = o.z + B3 == L3 ? 0 : o.z + B3;
            const int c4 = sb + o.z;
            // regions in the order the consumers release them: x3 faces, x2 faces, x1 faces, centre
            if (g >= 2) mbar_wait(eb, epar);
            mbar_arrive_expect_tx(bar, 2 * B1 * B2 * Cfg::ROWB);
            tma_load_5d_hint(dst + Cfg::R_X3M * Cfg::ROWB, &map_x3, bar, 0, 0, o.x, o.y, sb + x3m, pol_last);
            tma_load_5d_hint(dst + Cfg::R_X3P * Cfg::ROWB, &map_x3, bar, 0, 0, o.x, o.y, sb + x3p, pol_last);
            if (g >= 2) mbar_wait(eb + 8, epar);
            mbar_arrive_expect_tx(bar, 2 * B1 * B3 * Cfg::ROWB);
            tma_load_5d_hint(dst + Cfg::R_X2M * Cfg::ROWB, &map_x2, bar, 0, 0, o.x, x2m, c4, pol_last);
            tma_load_5d_hint(dst + Cfg::R_X2P * Cfg::ROWB, &map_x2, bar, 0, 0, o.x, x2p, c4, pol_last);
            if (g >= 2) mbar_wait(eb + 16, epar);
            mbar_arrive_expect_tx(bar, 2 * B2 * B3 * Cfg::ROWB);
            tma_load_5d_hint(dst + Cfg::R_X1M * Cfg::ROWB, &map_x1, bar, 0, 0, x1m, o.y, c4, pol_last);
            tma_load_5d_hint(dst + Cfg::R_X1P * Cfg::ROWB, &map_x1, bar, 0, 0, x1p, o.y, c4, pol_last);
            if (g >= 2) mbar_wait(eb + 24, epar);
            mbar_arrive_expect_tx(bar, Cfg::NROW_C * Cfg::ROWB);
            tma_load_5d_hint(dst, &map_c, bar, 0, 0, o.x, o.y, c4, pol_last);
        }
        }
        if constexpr (TM) {     // warp 0 frees the tensor memory once every consumer warp is done with it
            __syncwarp();
            asm volatile("bar.sync 2, %0;" ::"n"((Cfg::NWARP_C + 1) * 32) : "memory");
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512) : "memory");
        }
        return;
    }

    reg_alloc<Cfg::CONS_REGS>();
    const int ctid = tid - 128;
    if (ctid >= 3 * Cfg::TP) return;
    const int c = ctid / Cfg::TP, site = ctid % Cfg::TP;         // colour-major: uniform per warp
    double nsum = 0.0;
    consume64<LH, B1, B2, B3, MODE, TM>(args, smem, full_base, empty_base, exch_base, site, c, my_tiles, nsum, tmem_base);

    if constexpr ((MODE & 4) != 0) {
        // lanes -> warp (xor butterfly), warps -> CTA in warp order: the same order in every run
        double v = nsum;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        double *slots = reinterpret_cast<double *>(smem + Cfg::NSTAGE * Cfg::STAGE_BYTES + Cfg::RED_BYTES + Cfg::TAIL_NORM);
        if ((ctid & 31) == 0) slots[ctid >> 5] = v;
        asm volatile("bar.sync 1, %0;" ::"n"(Cfg::NWARP_C * 32) : "memory");      // consumer warps only
        if (ctid == 0) {
            double t = 0.0;
            for (int w = 0; w < Cfg::NWARP_C; w++) t += slots[w];
            args.norm_partials[blockIdx.x] = t;
        }
    }
    if constexpr (TM) {
        tmem_fence_before();
        asm volatile("bar.sync 2, %0;" ::"n"((Cfg::NWARP_C + 1) * 32) : "memory");
    }
}

// =============================================================================================
// Site-per-thread TMEM variant ("S"): ONE thread per output site, as in the fp32 kernel, with all 8 links of the
// site (72 complex = 288 words) parked in the thread's tensor-memory lane instead of in registers.  No colour split:
// no repeated accumulation (840 instead of 1248 fp64 operations per site), no exchange, no exchange barriers.
// Three warpgroups per CTA:
//   warps 0-3   link loaders: thread <-> site of the tile; write the NEXT tile's links into tensor memory while the
//               consumers compute (global -> registers -> tcgen05.st)
//   warps 4-7   consumers: 128 sites, one warp per TMEM lane quadrant (and per scheduler).  The link of leg L + 1 is
//               requested from tensor memory right after leg L's has been unpacked and lands during leg L's arithmetic
//   warp 8      producer: one thread issues the bulk tensor loads, region by region (warps 9-11 exit)
// Loader warp q and consumer warp q address the same 32 TMEM lanes (tcgen05.ld / .st reach lane quadrant warp % 4).
// A lane's 512 columns are 14 link slots of 36 columns (9 complex numbers U_ab at a*3 + b); the slot assignment and the
// four mbarriers per quadrant that hand slots back and forth are described at Staged64SCfg::NSLOT and in the kernel.
// =============================================================================================
template <int LH, int B1, int B2, int B3> struct Staged64SCfg {
    static constexpr int NROW_C = B1 * B2 * B3;
    static constexpr int T = LH * NROW_C;                        // output sites per tile (<= 128: one per TMEM lane)
    static constexpr int NWARP_C = 4;                            // consumer warps of the CTA
    static constexpr int NWARP_ACT = (T + 31) / 32;              // ... that own sites (row lengths that do not divide 128)
    // warpgroup 0: link loaders (one thread per site), warpgroup 1: consumers (one thread per site),
    // warpgroup 2: its first warp issues the bulk tensor loads
    static constexpr int NT = 384;
    // register split (setmaxnreg): the loaders keep the 168 of the launch, the producer warpgroup gives up what the
    // consumers take
    static constexpr int CONS_REGS = 256, PROD_REGS = 40;
    static constexpr int ROWB = 12 * LH * 16;
    static constexpr int R_X1M = NROW_C, R_X1P = R_X1M + B2 * B3, R_X2M = R_X1P + B2 * B3,
                         R_X2P = R_X2M + B1 * B3, R_X3M = R_X2P + B1 * B3, R_X3P = R_X3M + B1 * B2,
                         NROW_IN = R_X3P + B1 * B2;
    static constexpr int STAGE_BYTES = NROW_IN * ROWB;
    static constexpr int NSTAGE = 2;
    // regions of a stage, in the order the consumers finish with them: x3 faces, x2 faces, x1 faces, centre
    static constexpr int NREG = 4;
    // tensor memory: 14 slots of 36 columns (one link each).  Tile number t of a CTA keeps the link of the leg at
    // position p of the leg order (6 7 4 5 2 3 0 1) in slot (8 t + p) mod 14: the first six links of the next tile go
    // into the six slots this tile does not use, the last two into the slots of this tile's first two legs.
    static constexpr int NSLOT = 14;
    // tail: full[2] (16 B), empty[2][4] (64 B), four link barriers per lane quadrant (128 B: ready, early, free, done),
    // TMEM base (8 B), one fp64 slot per consumer warp (fused norm2)
    static constexpr int TAIL_LINK = 80, TAIL_TMEM = 208, TAIL_NORM = 216, TAIL = TAIL_NORM + 8 * NWARP_C;
    static constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + (TAIL + 15) / 16 * 16;
    static_assert(T <= 128 && T > 64, "one site per TMEM lane, one consumer warp per lane quadrant: 65..128 sites per tile");
    static_assert(SMEM_BYTES <= 232448, "tile too large for shared memory");
};

// the 36 words of one link: an x32 and an x4 load
__device__ __forceinline__ void tmem_ld36(uint32_t taddr, uint32_t (&r)[36])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]),
                   "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]),
                   "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr));
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r[32]), "=r"(r[33]), "=r"(r[34]), "=r"(r[35]) : "r"(taddr + 32));
}
__device__ __forceinline__ void tmem_wait_ld_regs36(uint32_t (&r)[36])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]), "+r"(r[9]), "+r"(r[10]),
                   "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15]), "+r"(r[16]), "+r"(r[17]), "+r"(r[18]), "+r"(r[19]), "+r"(r[20]),
                   "+r"(r[21]), "+r"(r[22]), "+r"(r[23]), "+r"(r[24]), "+r"(r[25]), "+r"(r[26]), "+r"(r[27]), "+r"(r[28]), "+r"(r[29]), "+r"(r[30]),
                   "+r"(r[31]), "+r"(r[32]), "+r"(r[33]), "+r"(r[34]), "+r"(r[35]));
}

// one whole leg for one site: acc += reconstruct( U * project(psi) ), psi[spin][colour], U[a*3 + b], acc[spin*3 + colour]
template <int MU, bool FWD, bool FIRST>
__device__ __forceinline__ void leg64_site(double2 (&acc)[12], const double2 (&psi)[4][3], const double2 (&U)[9])
{
    double2 h[2][3];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if constexpr (MU == 0) {
            h[0][c] = FWD ? csubi(psi[0][c], psi[3][c]) : caddi(psi[0][c], psi[3][c]);
            h[1][c] = FWD ? csubi(psi[1][c], psi[2][c]) : caddi(psi[1][c], psi[2][c]);
        } else if constexpr (MU == 1) {
            h[0][c] = FWD ? cadd(psi[0][c], psi[3][c]) : csub(psi[0][c], psi[3][c]);
            h[1][c] = FWD ? csub(psi[1][c], psi[2][c]) : cadd(psi[1][c], psi[2][c]);
        } else if constexpr (MU == 2) {
            h[0][c] = FWD ? csubi(psi[0][c], psi[2][c]) : caddi(psi[0][c], psi[2][c]);
            h[1][c] = FWD ? caddi(psi[1][c], psi[3][c]) : csubi(psi[1][c], psi[3][c]);
        } else {
            h[0][c] = FWD ? csub(psi[0][c], psi[2][c]) : cadd(psi[0][c], psi[2][c]);
            h[1][c] = FWD ? csub(psi[1][c], psi[3][c]) : cadd(psi[1][c], psi[3][c]);
        }
    }
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const double2 x0 = cmac(cmac(cmul(U[3 * a], h[0][0]), U[3 * a + 1], h[0][1]), U[3 * a + 2], h[0][2]);
        const double2 x1 = cmac(cmac(cmul(U[3 * a], h[1][0]), U[3 * a + 1], h[1][1]), U[3 * a + 2], h[1][2]);
        if constexpr (FIRST) {
            acc[0 + a] = x0;
            acc[3 + a] = x1;
            if constexpr (MU == 0) {
                acc[6 + a] = FWD ? cmuli(x1) : cmulni(x1);
                acc[9 + a] = FWD ? cmuli(x0) : cmulni(x0);
            } else if constexpr (MU == 1) {
                acc[6 + a] = FWD ? cneg(x1) : x1;
                acc[9 + a] = FWD ? x0 : cneg(x0);
            } else if constexpr (MU == 2) {
                acc[6 + a] = FWD ? cmuli(x0) : cmulni(x0);
                acc[9 + a] = FWD ? cmulni(x1) : cmuli(x1);
            } else {
                acc[6 + a] = FWD ? cneg(x0) : x0;
                acc[9 + a] = FWD ? cneg(x1) : x1;
            }
        } else {
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
}

template <int LH, int B1, int B2, int B3, int MODE>
__global__ void __launch_bounds__(Staged64SCfg<LH, B1, B2, B3>::NT, 1)
dhop_staged64s_kernel(const __grid_constant__ CUtensorMap map_c, const __grid_constant__ CUtensorMap map_x1,
                      const __grid_constant__ CUtensorMap map_x2, const __grid_constant__ CUtensorMap map_x3,
                      const Staged64Args args)
{
    using Cfg = Staged64SCfg<LH, B1, B2, B3>;
    constexpr bool DAG = (MODE & 1) != 0, AXPY = (MODE & 2) != 0, NORM = (MODE & 4) != 0;
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t full_base = smem_base + Cfg::NSTAGE * Cfg::STAGE_BYTES;        // full[2]
    const uint32_t empty_base = full_base + 16;                                   // empty[2][4]
    const uint32_t link_base = full_base + Cfg::TAIL_LINK;                        // [quadrant][ready, early, free, done]
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + Cfg::NSTAGE * Cfg::STAGE_BYTES + Cfg::TAIL_TMEM);
    const int tid = threadIdx.x;
    const int my_tiles = (args.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int nsteps = my_tiles * args.Ls;
    if (nsteps <= 0) {
        if (NORM && tid == 0) args.norm_partials[blockIdx.x] = 0.0;
        return;
    }
    if (tid == 0) {
        for (int i = 0; i < 2; i++) {
            mbar_init(full_base + 8 * i, Cfg::NREG);           // one arrive.expect_tx per region
            for (int r = 0; r < Cfg::NREG; r++) mbar_init(empty_base + 8 * (Cfg::NREG * i + r), Cfg::NWARP_ACT);
        }
        for (int i = 0; i < 16; i++) mbar_init(link_base + 8 * i, 1);
        mbar_fence_init();
    }
    if (tid >= 256 && tid < 288) {      // the producer warp allocates the tensor memory (one CTA per SM: all 512 columns)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tmem_fence_before();
    __syncthreads();
    tmem_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (tid >= 256) {       // ===================== producer: one thread issues the seven boxes of every step =====
        reg_dealloc<Cfg::PROD_REGS>();
        if (tid >= 288) return;
        if (tid == 256) {
            tma_prefetch_desc(&map_c);
            tma_prefetch_desc(&map_x1);
            tma_prefetch_desc(&map_x2);
            tma_prefetch_desc(&map_x3);
            const int L1 = args.L1, L2 = args.L2, L3 = args.L3;
            const uint64_t pol_last = l2_policy(args.l2pol % 10);
            for (int g = 0; g < nsteps; g++) {
                const int it = g / args.Ls, i = g % args.Ls, stage = g & 1;
                const int s = (args.zigzag && (it & 1)) ? args.Ls - 1 - i : i;
                const int4 o = args.tiles[blockIdx.x + it * gridDim.x];
                const uint32_t bar = full_base + 8 * stage;
                const uint32_t dst = smem_base + stage * Cfg::STAGE_BYTES;
                const int sb = s * L3;
                const int x1m = o.x == 0 ? L1 - 1 : o.x - 1, x1p = o.x + B1 == L1 ? 0 : o.x + B1;
                const int x2m = o.y == 0 ? L2 - 1 : o.y - 1, x2p = o.y + B2 == L2 ? 0 : o.y + B2;
                const int x3m = o.z == 0 ? L3 - 1 : o.z - 1, x3p = o.z + B3 == L3 ? 0 : o.z + B3;
                const int c4 = sb + o.z;
                // every region is refilled as soon as the four consumer warps have handed it back
                const uint32_t eb = empty_base + 8 * Cfg::NREG * stage;
                const uint32_t ph = ((g >> 1) - 1) & 1;
                if (g >= 2) mbar_wait(eb, ph);
                mbar_arrive_expect_tx(bar, 2 * B1 * B2 * Cfg::ROWB);
                tma_load_5d_hint(dst + Cfg::R_X3M * Cfg::ROWB, &map_x3, bar, 0, 0, o.x, o.y, sb + x3m, pol_last);
                tma_load_5d_hint(dst + Cfg::R_X3P * Cfg::ROWB, &map_x3, bar, 0, 0, o.x, o.y, sb + x3p, pol_last);
                if (g >= 2) mbar_wait(eb + 8, ph);
                mbar_arrive_expect_tx(bar, 2 * B1 * B3 * Cfg::ROWB);
                tma_load_5d_hint(dst + Cfg::R_X2M * Cfg::ROWB, &map_x2, bar, 0, 0, o.x, x2m, c4, pol_last);
                tma_load_5d_hint(dst + Cfg::R_X2P * Cfg::ROWB, &map_x2, bar, 0, 0, o.x, x2p, c4, pol_last);
                if (g >= 2) mbar_wait(eb + 16, ph);
                mbar_arrive_expect_tx(bar, 2 * B2 * B3 * Cfg::ROWB);
                tma_load_5d_hint(dst + Cfg::R_X1M * Cfg::ROWB, &map_x1, bar, 0, 0, x1m, o.y, c4, pol_last);
                tma_load_5d_hint(dst + Cfg::R_X1P * Cfg::ROWB, &map_x1, bar, 0, 0, x1p, o.y, c4, pol_last);
                if (g >= 2) mbar_wait(eb + 24, ph);
                mbar_arrive_expect_tx(bar, Cfg::NROW_C * Cfg::ROWB);
                tma_load_5d_hint(dst, &map_c, bar, 0, 0, o.x, o.y, c4, pol_last);
            }
        }
        __syncwarp();       // this warp frees the tensor memory once the loaders and the consumers are done with it
        asm volatile("bar.sync 2, %0;" ::"n"(288) : "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512) : "memory");
        return;
    }

    // loaders and consumers: thread <-> site of the tile, warp <-> TMEM lane quadrant.  Tiles of fewer than 128 sites
    // (row lengths 12, 20, 24, 28): a warp without sites idles; the lanes without a site in the last active warp run
    // along on the tile's last site (the warp-wide tcgen05 instructions need every lane) and do not store.
    const int site_raw = tid & 127;
    const bool warp_act = (site_raw & ~31) < Cfg::T, lane_act = site_raw < Cfg::T;
    const int site = lane_act ? site_raw : Cfg::T - 1;
    const int h = site % LH, row = site / LH;
    const int i1 = row % B1, i2 = (row / B1) % B2, i3 = row / (B1 * B2);
    const int lane = tid & 31, quad = site_raw >> 5;
    const uint32_t tm_links = tmem_base + ((uint32_t)(quad * 32) << 16);
    const uint32_t bar_ready = link_base + 32 * quad, bar_early = bar_ready + 8, bar_free = bar_ready + 16, bar_done = bar_ready + 24;
    auto tile_row = [&](int it, int &r) -> long long {
        const int4 o = args.tiles[blockIdx.x + it * gridDim.x];
        const int x1 = o.x + i1, x2 = o.y + i2, x3 = o.z + i3;
        r = (x1 + x2 + x3 + args.parity_out) & 1;
        return x1 + (long long)args.L1 * (x2 + (long long)args.L2 * x3);
    };
    // TMEM column of the link at position p (0..7) of the leg order for the tile whose slot base is b8 = (8 t) mod 14
    auto slot_col = [&](int b8, int p) -> uint32_t {
        int sl = b8 + p;
        if (sl >= Cfg::NSLOT) sl -= Cfg::NSLOT;
        return 36u * (uint32_t)sl;
    };

    if (tid < 128) {        // ===================== link loaders: global -> tensor memory, one tile ahead ============
        const uint64_t pol_first = l2_policy(args.l2pol / 1000000 % 10);
        int b8 = 0;
        for (int n = 0; warp_act && n < my_tiles; n++) {
            int r_unused;
            const long long grow = tile_row(n, r_unused);
            const double2 *gp = args.gauge + grow * (72 * LH) + 2 * h;
            // position p of the leg order holds leg (6 - 2 (p / 2)) + (p & 1): elements [9 leg, 9 leg + 9) of the site.
            // Elements 2j and 2j + 1 are adjacent in memory (pack.cu): 256-bit loads, whole 512-byte runs per warp.
            // Two batches of 18 elements (72 registers each) are in flight at a time.
            double2 ta[18], tb[18];
#pragma unroll
            for (int k = 0; k < 18; k += 2) ldg_d4_hint(gp + (54 + k) * LH, pol_first, ta[k], ta[k + 1]);      // legs 6, 7
#pragma unroll
            for (int k = 0; k < 18; k += 2) ldg_d4_hint(gp + (36 + k) * LH, pol_first, tb[k], tb[k + 1]);      // legs 4, 5
            // the slots of positions 0..5 were last read by tile n - 2 (n >= 2)
            if (n >= 2) {
                mbar_wait(bar_done, (n - 2) & 1);
                tmem_fence_after();
            }
#pragma unroll
            for (int k = 0; k < 18; k++) tmem_st_c(tm_links + slot_col(b8, 0 + k / 9) + 4 * (k % 9), ta[k]);
#pragma unroll
            for (int k = 0; k < 18; k += 2) ldg_d4_hint(gp + (18 + k) * LH, pol_first, ta[k], ta[k + 1]);      // legs 2, 3
#pragma unroll
            for (int k = 0; k < 18; k++) tmem_st_c(tm_links + slot_col(b8, 2 + k / 9) + 4 * (k % 9), tb[k]);
#pragma unroll
            for (int k = 0; k < 18; k += 2) ldg_d4_hint(gp + k * LH, pol_first, tb[k], tb[k + 1]);             // legs 0, 1
#pragma unroll
            for (int k = 0; k < 18; k++) tmem_st_c(tm_links + slot_col(b8, 4 + k / 9) + 4 * (k % 9), ta[k]);
            tmem_wait_st();
            tmem_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_early);
            // the slots of positions 6, 7 are those of the first two legs of tile n - 1: free once its last slice has
            // taken them into registers
            if (n >= 1) {
                mbar_wait(bar_free, (n - 1) & 1);
                tmem_fence_after();
            }
#pragma unroll
            for (int k = 0; k < 18; k++) tmem_st_c(tm_links + slot_col(b8, 6 + k / 9) + 4 * (k % 9), tb[k]);
            tmem_wait_st();
            tmem_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_ready);
            b8 = (b8 + 8) % Cfg::NSLOT;
        }
        asm volatile("bar.sync 2, %0;" ::"n"(288) : "memory");
        return;
    }

    // =========================== consumers: one thread = one output site ===========================
    reg_alloc<Cfg::CONS_REGS>();
    const uint64_t pol_out = l2_policy(args.l2pol / 10000000 % 10);
    const int rc = row;
    const int r1p = (i1 + 1 < B1) ? rc + 1 : Cfg::R_X1P + i2 + B2 * i3;
    const int r1m = (i1 > 0) ? rc - 1 : Cfg::R_X1M + i2 + B2 * i3;
    const int r2p = (i2 + 1 < B2) ? rc + B1 : Cfg::R_X2P + i1 + B1 * i3;
    const int r2m = (i2 > 0) ? rc - B1 : Cfg::R_X2M + i1 + B1 * i3;
    const int r3p = (i3 + 1 < B3) ? rc + B1 * B2 : Cfg::R_X3P + i1 + B1 * i2;
    const int r3m = (i3 > 0) ? rc - B1 * B2 : Cfg::R_X3M + i1 + B1 * i2;
    uint32_t off[8];            // byte offsets of (neighbour site, component 0) inside a stage; component k at + k * KB
    constexpr uint32_t KB = LH * 16;
    off[2] = r1p * Cfg::ROWB + h * 16;
    off[3] = r1m * Cfg::ROWB + h * 16;
    off[4] = r2p * Cfg::ROWB + h * 16;
    off[5] = r2m * Cfg::ROWB + h * 16;
    off[6] = r3p * Cfg::ROWB + h * 16;
    off[7] = r3m * Cfg::ROWB + h * 16;
    const long long nrow = (long long)args.L1 * args.L2 * args.L3;
    auto set_x0_offsets = [&](int r) {
        int hp = h + r;       if (hp == LH) hp = 0;
        int hm = h - 1 + r;   if (hm < 0) hm = LH - 1;
        off[0] = rc * Cfg::ROWB + hp * 16;
        off[1] = rc * Cfg::ROWB + hm * 16;
    };

    double nsum = 0.0;
    int g = 0, b8 = 0;
    for (int it = 0; warp_act && it < my_tiles; it++) {
        const bool has_next = it + 1 < my_tiles;
        int r_cur;
        const long long grow = tile_row(it, r_cur);
        set_x0_offsets(r_cur);
        const uint32_t tm_tile = tm_links + 36u * (uint32_t)b8;
        // TMEM address of the link at position p of this tile (slots wrap at 14)
#define DWF_LINK_AT(p) (tm_tile + ((b8 + (p)) >= Cfg::NSLOT ? (uint32_t)(36 * (p)) - 36u * Cfg::NSLOT : (uint32_t)(36 * (p))))
        mbar_wait(bar_ready, it & 1);           // the loader warp of this lane quadrant has written all eight links
        tmem_fence_after();
        for (int ss = 0; ss < args.Ls; ss++, g++) {
            const int s = (args.zigzag && (it & 1)) ? args.Ls - 1 - ss : ss;
            const int stage = g & 1;
            const bool hand_over = has_next && ss == args.Ls - 1;
            double2 *o2 = args.out + grow * (12 * LH) + h + (long long)s * nrow * (12 * LH);
            mbar_wait(full_base + 8 * stage, (g >> 1) & 1);
            const unsigned char *sb = smem + stage * Cfg::STAGE_BYTES;
            double2 acc[12];
            uint32_t W[36];
            tmem_ld36(DWF_LINK_AT(0), W);
            double2 xv[12];
            // one leg: the neighbour spinor out of shared memory, the link out of tensor memory (requested one leg
            // ahead: right after this leg's link has been unpacked, the next one's load goes into the same registers)
#define DWF_LEG64S(L, MU, FWD, FIRST, NEXTP)                                                        \
            {                                                                                       \
                double2 psi[4][3];                                                                  \
                _Pragma("unroll") for (int k = 0; k < 12; k++)                                      \
                    psi[k / 3][k % 3] = *reinterpret_cast<const double2 *>(sb + off[L] + k * KB);   \
                tmem_wait_ld_regs36(W);                                                             \
                double2 Ul[9];                                                                      \
                _Pragma("unroll") for (int k = 0; k < 9; k++) Ul[k] = tmem_unpack_p(W + 4 * k);     \
                if constexpr ((NEXTP) >= 0) tmem_ld36(DWF_LINK_AT((NEXTP) < 0 ? 0 : (NEXTP)), W);   \
                leg64_site<MU, (FWD) != DAG, FIRST>(acc, psi, Ul);                                  \
            }
            // a region goes back to the producer as soon as this warp's loads from it have completed: the accumulator
            // rows acc[0], acc[3] (spin 0 and 1, colour 0) derive from all twelve components of every neighbour read
            // so far, and the arrive's address is computed from them (tma.cuh, mbar_arrive_dep)
#define DWF_RELEASE64S(R)                                                                           \
            __syncwarp();                                                                           \
            if (lane == 0) mbar_arrive_dep(empty_base + 8 * (Cfg::NREG * stage + (R)), args.zero, acc[0].x, acc[3].x);
            DWF_LEG64S(6, 3, true, true, 1)
            DWF_LEG64S(7, 3, false, false, 2)
            DWF_RELEASE64S(0)
            if (hand_over) {
                // last slice of the tile: the links of its first two legs are in registers (tcgen05.wait::ld inside the
                // leg), their slots go to the loader for the next tile's last two links.  The wait on `early` keeps
                // this warp at most one phase ahead of the loader on `free` and `done`.
                mbar_wait(bar_early, (it + 1) & 1);
                tmem_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_free);
            }
            DWF_LEG64S(4, 2, true, false, 3)
            DWF_LEG64S(5, 2, false, false, 4)
            DWF_RELEASE64S(1)
            DWF_LEG64S(2, 1, true, false, 5)
            DWF_LEG64S(3, 1, false, false, 6)
            DWF_RELEASE64S(2)
            DWF_LEG64S(0, 0, true, false, 7)
            if constexpr (AXPY) {       // x of this site and slice, requested before the last leg
                const double2 *xp = args.axpy_x + (o2 - args.out);
#pragma unroll
                for (int k = 0; k < 12; k++) xv[k] = lane_act ? __ldcs(xp + k * LH) : make_double2(0.0, 0.0);
            }
            DWF_LEG64S(1, 0, false, false, -1)
#undef DWF_LEG64S
            DWF_RELEASE64S(3)
#undef DWF_RELEASE64S
            if (ss == args.Ls - 1) {    // every link of this tile has been read for the last time
                tmem_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_done);
            }
#pragma unroll
            for (int k = 0; k < 12; k++) {
                double2 v = acc[k];
                if constexpr (AXPY) {
                    v.x = fma(args.axpy_b, v.x, args.axpy_a * xv[k].x);
                    v.y = fma(args.axpy_b, v.y, args.axpy_a * xv[k].y);
                }
                if (lane_act) {
                    if constexpr (NORM) nsum = fma(v.x, v.x, fma(v.y, v.y, nsum));
                    stg_d2_hint(o2 + k * LH, v, pol_out);
                }
            }
        }
#undef DWF_LINK_AT
        b8 = (b8 + 8) % Cfg::NSLOT;
    }

    if constexpr (NORM) {
        double v = nsum;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        double *slots = reinterpret_cast<double *>(smem + Cfg::NSTAGE * Cfg::STAGE_BYTES + Cfg::TAIL_NORM);
        if (lane == 0) slots[quad] = v;
        asm volatile("bar.sync 1, %0;" ::"n"(Cfg::NWARP_C * 32) : "memory");
        if (site == 0) {
            double t = 0.0;
            for (int w = 0; w < Cfg::NWARP_C; w++) t += slots[w];
            args.norm_partials[blockIdx.x] = t;
        }
    }
    tmem_fence_before();
    asm volatile("bar.sync 2, %0;" ::"n"(288) : "memory");
}

// ---------------------------------------------------------------------------------------------
// Kernel instances: this file is compiled once per MODE (-DDWF_STAGED64_MODE=0..4, build.py); each
// translation unit exports the entry points of its MODE in the order of DWF_STAGED64_VARIANTS, the
// MODE 0 unit also holds the host code.
// ---------------------------------------------------------------------------------------------
#define DWF_STAGED64_VARIANTS(X) X(16, 2, 1, 2) X(16, 1, 1, 4) X(16, 1, 2, 2) X(16, 2, 2, 1) X(8, 4, 2, 1) X(8, 2, 2, 2) X(4, 4, 4, 1) X(4, 4, 2, 2) X(4, 2, 2, 2) X(4, 2, 2, 1) X(8, 2, 2, 1) X(16, 2, 1, 1) \
    X(12, 2, 1, 2) X(12, 2, 2, 1) X(12, 1, 2, 2) X(24, 2, 1, 1) X(24, 1, 1, 2) X(32, 2, 1, 1) X(32, 1, 1, 2) X(32, 1, 2, 1) X(20, 1, 1, 2) X(20, 2, 1, 1)

// TMEM variants (128-site tiles), preferred when they fit the lattice
#define DWF_STAGED64T_VARIANTS(X) X(16, 2, 2, 2) X(8, 4, 2, 2) X(8, 2, 4, 2) X(8, 2, 2, 4) X(4, 4, 4, 2) X(4, 4, 2, 4)
// site-per-thread TMEM variants: the 128-site shapes plus 96 .. 120-site tiles for the row lengths that do not divide 128
#define DWF_STAGED64S_VARIANTS(X) DWF_STAGED64T_VARIANTS(X) X(12, 2, 2, 2) X(24, 2, 2, 1) X(24, 1, 2, 2) X(24, 2, 1, 2) \
    X(20, 3, 2, 1) X(20, 1, 2, 3) X(28, 2, 2, 1) X(28, 1, 2, 2)

const void *const *staged64_kernels_mode0();
const void *const *staged64_kernels_mode1();
const void *const *staged64_kernels_mode2();
const void *const *staged64_kernels_mode3();
const void *const *staged64_kernels_mode4();

#define DWF_CAT2(a, b) a##b
#define DWF_CAT(a, b) DWF_CAT2(a, b)
const void *const *DWF_CAT(staged64_kernels_mode, DWF_STAGED64_MODE)()
{
#define X(LH, B1, B2, B3) reinterpret_cast<const void *>(&dhop_staged64_kernel<LH, B1, B2, B3, DWF_STAGED64_MODE, true>),
#define Y(LH, B1, B2, B3) reinterpret_cast<const void *>(&dhop_staged64_kernel<LH, B1, B2, B3, DWF_STAGED64_MODE, false>),
#define Z(LH, B1, B2, B3) reinterpret_cast<const void *>(&dhop_staged64s_kernel<LH, B1, B2, B3, DWF_STAGED64_MODE>),
    // order of preference: site-per-thread TMEM kernels, colour-split TMEM kernels, colour-split register kernels
    static const void *const tab[] = {DWF_STAGED64S_VARIANTS(Z) DWF_STAGED64T_VARIANTS(X) DWF_STAGED64_VARIANTS(Y)};
#undef X
#undef Y
#undef Z
    return tab;
}

#if DWF_STAGED64_MODE == 0
// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct Variant64 {
    int lh, b1, b2, b3, smem, threads, tmem;
    const void *fn[5];       // MODE 0 plain, 1 dagger, 2 a x + b Dhop, 3 a x + b Dhop^dagger, 4 Dhop + norm2
};

static const std::vector<Variant64> &variants64()
{
    static const std::vector<Variant64> v = [] {
        std::vector<Variant64> t;
        const void *const *k0 = staged64_kernels_mode0(), *const *k1 = staged64_kernels_mode1(), *const *k2 = staged64_kernels_mode2(),
                          *const *k3 = staged64_kernels_mode3(), *const *k4 = staged64_kernels_mode4();
#define X(LH, B1, B2, B3)                                                                             \
        t.push_back({LH, B1, B2, B3, Staged64SCfg<LH, B1, B2, B3>::SMEM_BYTES, Staged64SCfg<LH, B1, B2, B3>::NT, 2, \
                     {k0[t.size()], k1[t.size()], k2[t.size()], k3[t.size()], k4[t.size()]}});
        DWF_STAGED64S_VARIANTS(X)
#undef X
#define X(LH, B1, B2, B3)                                                                             \
        t.push_back({LH, B1, B2, B3, Staged64Cfg<LH, B1, B2, B3, true>::SMEM_BYTES, Staged64Cfg<LH, B1, B2, B3, true>::NT, 1, \
                     {k0[t.size()], k1[t.size()], k2[t.size()], k3[t.size()], k4[t.size()]}});
        DWF_STAGED64T_VARIANTS(X)
#undef X
#define X(LH, B1, B2, B3)                                                                             \
        t.push_back({LH, B1, B2, B3, Staged64Cfg<LH, B1, B2, B3>::SMEM_BYTES, Staged64Cfg<LH, B1, B2, B3>::NT, 0, \
                     {k0[t.size()], k1[t.size()], k2[t.size()], k3[t.size()], k4[t.size()]}});
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
        g->staged64.kind = v[i].tmem;
        g->staged64.b[0] = v[i].b1; g->staged64.b[1] = v[i].b2; g->staged64.b[2] = v[i].b3;
        g->staged64.ntiles = (lat.L[1] / v[i].b1) * (lat.L[2] / v[i].b2) * (lat.L[3] / v[i].b3);
        // per-device opt-in to the large dynamic shared memory (the caller holds a DeviceGuard)
        for (int d = 0; d < 5; d++)
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
static int encode_map64(CUtensorMap *m, const void *base, const Lattice &lat, int Ls, int b1, int b2, int b3)
{
    PFN_tensorMapEncodeTiled enc = get_tensor_map_encoder();
    const cuuint64_t dims[5] = {(cuuint64_t)2 * lat.Lh, 12, (cuuint64_t)lat.L[1], (cuuint64_t)lat.L[2],
                                (cuuint64_t)lat.L[3] * Ls};
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

// The four tensor maps of a field depend on its pointer and the tile shape only: kept in a small
// per-thread cache (keyed by geometry id, variant and pointer) so that a solver that applies the
// operator to the same few buffers makes no driver calls (as dhop_staged.cu does for fp32).
struct MapSet64 { unsigned long long gid; int variant, ls; const void *ptr; CUtensorMap m[4]; };

static int get_maps64(const dwf_geometry *g, const Variant64 &v, const void *ptr, int ls, const MapSet64 **out)
{
    static thread_local MapSet64 cache[8];
    static thread_local unsigned next_slot = 0;
    for (const MapSet64 &c : cache)
        if (c.ptr == ptr && c.gid == g->uid && c.variant == g->staged64.variant && c.ls == ls) { *out = &c; return DWF_OK; }
    MapSet64 t;
    t.gid = g->uid; t.variant = g->staged64.variant; t.ptr = ptr; t.ls = ls;
    int rc;
    if ((rc = encode_map64(&t.m[0], ptr, g->lat, ls, v.b1, v.b2, v.b3))) return rc;
    if ((rc = encode_map64(&t.m[1], ptr, g->lat, ls, 1, v.b2, v.b3))) return rc;
    if ((rc = encode_map64(&t.m[2], ptr, g->lat, ls, v.b1, 1, v.b3))) return rc;
    if ((rc = encode_map64(&t.m[3], ptr, g->lat, ls, v.b1, v.b2, 1))) return rc;
    MapSet64 *ms = &cache[next_slot++ % 8];
    *ms = t;
    *out = ms;
    return DWF_OK;
}

int launch_dhop_staged64(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st, bool dagger,
                         const void *axpy_x, double axpy_a, double axpy_b, double *norm_partials, int *norm_blocks, int nrhs)
{
    const int ls = g->lat.Ls * nrhs;       // nrhs fields one after the other = one field of nrhs * Ls slices (dhop_staged.cu)
    if (norm_partials && (dagger || axpy_x)) {
        set_error("the fp64 staged kernel has no instance for this combination of modes");
        return DWF_ERR_UNSUPPORTED;
    }
    const Variant64 &v = variants64()[(size_t)g->staged64.variant];
    const MapSet64 *ms = nullptr;
    int rc;
    if ((rc = get_maps64(g, v, in, ls, &ms))) return rc;
    CUtensorMap mc = ms->m[0], m1 = ms->m[1], m2 = ms->m[2], m3 = ms->m[3];     // passed by value
    Staged64Args a;
    a.out = static_cast<double2 *>(out);
    a.gauge = static_cast<const double2 *>(g->gauge[parity_out]);
    a.tiles = g->tiles_staged64;
    a.ntiles = g->staged64.ntiles;
    a.L1 = g->lat.L[1]; a.L2 = g->lat.L[2]; a.L3 = g->lat.L[3]; a.Ls = ls;
    a.parity_out = parity_out;
    a.zigzag = g->opt_zigzag;
    a.l2pol = g->opt_l2pol;
    a.zero = 0;
    a.axpy_x = static_cast<const double2 *>(axpy_x);
    a.axpy_a = axpy_a;
    a.axpy_b = axpy_b;
    a.norm_partials = norm_partials;
    const void *fn = v.fn[norm_partials ? 4 : (dagger ? 1 : 0) + (axpy_x ? 2 : 0)];
    const int grid_max = (g->opt_max_ctas > 0 && g->opt_max_ctas < g->sm_count) ? g->opt_max_ctas : g->sm_count;
    const int grid = g->staged64.ntiles < grid_max ? g->staged64.ntiles : grid_max;
    void *params[] = {&mc, &m1, &m2, &m3, &a};
    DWF_CUDA_CHECK(cudaLaunchKernel(fn, dim3((unsigned)grid), dim3((unsigned)v.threads), params, (size_t)v.smem, st));
    if (norm_blocks) *norm_blocks = grid;
    count_launch();
    return DWF_OK;
}

#endif  // DWF_STAGED64_MODE == 0

}  // namespace dwf

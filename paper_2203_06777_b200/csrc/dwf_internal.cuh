// dwf_internal.cuh -- shared declarations of libdwf's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include <stdio.h>
#include <atomic>

#include "../../include/dwf.h"

namespace dwf {

// ---------------------------------------------------------------------------------------------
// errors
// ---------------------------------------------------------------------------------------------
void set_error(const char *fmt, ...);
extern std::atomic<unsigned long long> g_launches;
inline void count_launch(int n = 1) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

#define DWF_CUDA_CHECK(expr)                                                                 \
    do {                                                                                     \
        cudaError_t e__ = (expr);                                                            \
        if (e__ != cudaSuccess) {                                                            \
            dwf::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, \
                           __LINE__);                                                        \
            return DWF_ERR_CUDA;                                                             \
        }                                                                                    \
    } while (0)

// ---------------------------------------------------------------------------------------------
// lattice description handed to kernels (by value, lives in the constant bank)
// ---------------------------------------------------------------------------------------------
struct Lattice {
    int L[4];        // extents, time last
    int Lh;          // L[0] / 2
    int Ls;
    long long V4;    // L0*L1*L2*L3
    long long Vh;    // V4 / 2
};

// How one CTA of the direct (L1-cached) kernel maps onto output sites.  A CTA owns a 4D tile of
// output sites of one parity (extents are powers of two; extent 0 counts x0-PAIRS) times `cpc`
// s-slices.
struct Tiling {
    int sh[4];       // log2 of the tile extents
    int ntile[4];    // tiles per direction
    int cpc;         // s-slices handled by one CTA
    int ncg;         // slice groups = Ls / cpc
    int threads;     // tile sites * cpc
    int ntiles;      // ntile[0]*ntile[1]*ntile[2]*ntile[3]
};

// Plan of the staged kernel (dhop_staged.cu): a CTA owns a box of B1 x B2 x B3 x0-rows (each row
// holds the Lh output sites of one parity of a lattice line along x0) and all Ls slices.
struct StagedPlan {
    int variant;     // index into the table of compiled (Lh, B1, B2, B3) instances, -1: not usable
    int kind;        // fp64 only: 0 colour split in registers, 1 colour split in tensor memory, 2 one thread per site, links in tensor memory
    int b[3];        // rows box
    int ntiles;
};

}  // namespace dwf

// the opaque handle of dwf.h
struct dwf_geometry {
    unsigned long long uid;  // unique per created geometry (never reused; keys the tensor-map cache)
    dwf::Lattice lat;
    int prec;               // DWF_F32 / DWF_F64
    int bc_time;
    int device;
    int sm_count;
    bool gauge_loaded;
    // device gauge: for each OUTPUT parity p the 8 links every output site needs,
    // planar over sites: [leg][18 reals in 128-bit vectors][cb site]; leg = 2*mu + (0: fwd, 1: bwd)
    void *gauge[2];
    size_t gauge_bytes;     // per parity
    // option "gauge12": rows 0, 1 of every link only (12 reals), [row][24 vectors][Lh]; fp32, used by the plain staged Dhop
    void *gauge12[2];
    int opt_gauge12;
    // U_t of the last time layer, per parity of the site, complex[row2][9][h]: the links the face kernels of halo.cu need
    // (in the packed sets the wrapping time links are sign-folded or, with DWF_OPEN_T, zero)
    void *tlink_top[2];
    // direct kernel: CTA tile table (origins in rasterised launch order)
    dwf::Tiling tiling_cb;
    int4 *tiles_cb;
    // staged (TMA, link-stationary) kernel: plan chosen at create time, row-box tile table
    dwf::StagedPlan staged;
    int4 *tiles_staged;
    // fp64 staged kernel (dhop_staged64.cu): its own tile shape and table
    dwf::StagedPlan staged64;
    int4 *tiles_staged64;
    // reductions
    double *partials;       // [2 * max_blocks]
    double *result_dev;     // [2]
    double *mailbox_host;   // mapped pinned host memory, MAILBOX_SLOTS slots of four words: [0..1] values, [2] sequence number of the reduction that wrote them
    double *mailbox_dev;    // the same words as the device sees them
    unsigned long long mailbox_seq;   // last sequence number handed to a reduction
    int reduce_blocks;
    // Host <-> device transfers of canonical arrays (dwf_import_spinor / dwf_export_spinor with host
    // buffers) go through a bounded ring: per direction (0: import, 1: export) one copy stream and two
    // device buffers of xfer_chunk bytes; the copy of chunk k+1 overlaps the reorder kernel of chunk k,
    // and the two directions use different streams (PCIe is full duplex).  Created on first use.
    struct HostXfer {
        bool ready;
        size_t chunk;                       // bytes per ring buffer
        cudaStream_t copy_stream[2];
        void *buf[2][2];
        cudaEvent_t filled[2][2];           // buffer holds a chunk (import: H2D done; export: reorder done)
        cudaEvent_t drained[2][2];          // buffer may be overwritten (import: reorder done; export: D2H done)
        unsigned long long count[2];        // chunks issued so far (ring position)
        // export reorder kernels run on their own stream behind an event of the caller's stream, so that the
        // caller's stream is not held up for the duration of the D2H copies; library calls that launch work
        // on a caller's stream first wait for export_done (they might overwrite the field being exported)
        cudaStream_t export_stream;
        cudaEvent_t export_begin, export_done;
        bool export_pending;
        const char *export_ptr;             // device field (and its size) an asynchronous export is still reading
        size_t export_bytes;
    } xfer;
    int opt_async_host;     // 1: host imports / exports return without synchronising (dwf_host_wait)
    int opt_full_launch;    // 1: dwf_dhop of a full fp32 field is one launch over both parities (0: two half launches)
    int opt_max_ctas;       // > 0: cap on the grid of the staged kernels (more tiles per CTA; tests of the tile switch)
    // tunables (dwf_set_option)
    int opt_tile[4];        // requested log2 tile extents (cb: dim 0 in pairs)
    int opt_cpc;
    int opt_raster;         // rasterisation order of the direct kernel's tile table
    int opt_raster_staged;  // ... of the staged kernel's tile table
    int opt_variant;        // restrict the staged kernel to one compiled variant (0: auto)
    int opt_kernel;         // 0: auto, 1: direct only, 2: staged only
    int opt_l2pol;          // staged kernel: L2 eviction-priority digits (dhop_staged.cu PC_*)
    int opt_ssplit;         // staged kernel: CTAs sharing one tile (each takes Ls / ssplit slices)
    int opt_zigzag;         // staged kernel: walk the slices of every other tile backwards
    int opt_layered;        // staged kernel: one TMA box per x3 layer, so that L2 policies can differ per layer
};

namespace dwf {

int rebuild_tilings(dwf_geometry *g);

// api.cu helpers used by the other translation units
constexpr unsigned long long MAILBOX_SLOTS = 8;
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
bool parity_ok(int p);
// orders later work on st that WRITES [written, written + bytes) behind the reorder kernels of an asynchronous
// host export still reading that memory (written == nullptr: any memory)
void wait_for_exports(const dwf_geometry *g, cudaStream_t st, const void *written = nullptr, size_t bytes = 0);
bool aligned16(const void *p);
// one half-Dhop (or a x + b Dhop) on the best kernel for the geometry
int half_dhop(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st, bool dagger = false,
              const void *axpy_x = nullptr, double a = 0.0, double b = 0.0, int nrhs = 1);
// waits for the reduction last enqueued on st and returns its n values (through the mapped mailbox)
int fetch_reduction(const dwf_geometry *g, cudaStream_t st, int n, double *out, unsigned long long seq = 0);     // seq 0: the reduction enqueued last

// pack.cu
int launch_pack_gauge(const dwf_geometry *g, const void *U_canonical_dev, cudaStream_t st);
int launch_compress_gauge12(const dwf_geometry *g, cudaStream_t st);      // gauge[p] -> gauge12[p]
// halo.cu
int launch_pack_tlinks(const dwf_geometry *g, const void *U_canonical_dev, cudaStream_t st);
// row0, nrow_c: lattice lines (rows) covered, nrow_c < 0 = the whole field; canonical_dev points at the first site of the range
int launch_import(const dwf_geometry *g, const void *canonical_dev, int parity, void *field,
                  cudaStream_t st, long long row0 = 0, long long nrow_c = -1);
int launch_export(const dwf_geometry *g, const void *field, int parity, void *canonical_dev,
                  cudaStream_t st, long long row0 = 0, long long nrow_c = -1);
// dhop.cu (direct kernel; half fields only)
int launch_dhop_direct(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st,
                       bool dagger = false, const void *axpy_x = nullptr, double axpy_a = 0.0, double axpy_b = 0.0);
// dhop_staged.cu (TMA-staged link-stationary kernel, fp32 half fields)
void plan_staged(dwf_geometry *g);                      // fills g->staged (variant = -1 if unusable)
void build_staged_tile_table(const dwf_geometry *g, int raster, int4 *host_table);
// norm_partials != nullptr: the fused-norm2 kernel writes one partial of |out|^2 per CTA there, *norm_blocks = their number
int launch_dhop_staged(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st,
                       double *norm_partials = nullptr, int *norm_blocks = nullptr, bool dagger = false,
                       const void *axpy_x = nullptr, float axpy_a = 0.f, float axpy_b = 0.f,     // axpy_x: out = a x + b Dhop in
                       int nrhs = 1,                                                            // nrhs fields one after the other
                       bool gauge12 = false,                                                    // 12-real links (plain Dhop only)
                       bool full = false,                                                       // in / out are full fields: one launch for both parities
                       bool half = false);                                                      // in / out are fp16-stored half fields
bool staged_supports_axpy(const dwf_geometry *g);
bool staged_supports_half(const dwf_geometry *g);       // a staged variant whose fp16 rows stay 128-byte aligned
// pack.cu: out = a x + b out, elementwise over nreal reals (the unfused path of dwf_dhop_*_axpy)
int launch_axpby(const dwf_geometry *g, const void *x, void *out, double a, double b, size_t nreal, cudaStream_t st);
// dhop_staged64.cu (TMA-staged fp64 kernel, links split by colour column over three threads)
void plan_staged64(dwf_geometry *g);
void build_staged64_tile_table(const dwf_geometry *g, int4 *host_table);
// norm_partials != nullptr: the fused-norm2 instance, one partial of |out|^2 per CTA, *norm_blocks = their number
int launch_dhop_staged64(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st, bool dagger,
                         const void *axpy_x = nullptr, double axpy_a = 0.0, double axpy_b = 0.0,
                         double *norm_partials = nullptr, int *norm_blocks = nullptr, int nrhs = 1);
// reduce.cu
int launch_norm2(const dwf_geometry *g, const void *field, size_t nreal, cudaStream_t st);
int launch_final_sum(const dwf_geometry *g, int nblocks, cudaStream_t st);   // result_dev[0] = sum of partials[0..nblocks)
int launch_inner(const dwf_geometry *g, const void *a, const void *b, size_t ncomplex,
                 cudaStream_t st);

}  // namespace dwf

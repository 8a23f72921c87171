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
    int Sc;          // s-slices per register block (device layout parameter)
    int nchunk;      // Ls / Sc
    long long V4;    // L0*L1*L2*L3
    long long Vh;    // V4 / 2
};

// How one CTA maps onto output sites.  A CTA owns a 4D tile of output sites (extents are
// powers of two; in checkerboard kernels extent 0 counts x0-PAIRS) times `cpc` s-chunks.
struct Tiling {
    int sh[4];       // log2 of the tile extents
    int ntile[4];    // tiles per direction
    int cpc;         // s-chunks handled by one CTA
    int ncg;         // chunk groups = nchunk / cpc
    int threads;     // tile sites * cpc
    int ntiles;      // ntile[0]*ntile[1]*ntile[2]*ntile[3]
};

}  // namespace dwf

// the opaque handle of dwf.h
struct dwf_geometry {
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
    // CTA tile tables (origins in rasterised launch order), one for cb kernels, one for full
    dwf::Tiling tiling_cb, tiling_full;
    int4 *tiles_cb, *tiles_full;
    // reductions
    double *partials;       // [2 * max_blocks]
    double *result_dev;     // [2]
    int reduce_blocks;
    // host-side staging for canonical <-> device conversions (lazily grown)
    void *staging;
    size_t staging_bytes;
    // tunables (dwf_set_option)
    int opt_tile[4];        // requested log2 tile extents (cb: dim 0 in pairs)
    int opt_cpc;
    int opt_raster;         // rasterisation order of the tile table
    int opt_variant;
};

namespace dwf {

int rebuild_tilings(dwf_geometry *g);

// pack.cu
int launch_pack_gauge(const dwf_geometry *g, const void *U_canonical_dev, cudaStream_t st);
int launch_import(const dwf_geometry *g, const void *canonical_dev, int parity, void *field,
                  cudaStream_t st);
int launch_export(const dwf_geometry *g, const void *field, int parity, void *canonical_dev,
                  cudaStream_t st);
// dhop.cu
int launch_dhop(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st);
// reduce.cu
int launch_norm2(const dwf_geometry *g, const void *field, size_t nreal, cudaStream_t st);
int launch_inner(const dwf_geometry *g, const void *a, const void *b, size_t ncomplex,
                 cudaStream_t st);

}  // namespace dwf

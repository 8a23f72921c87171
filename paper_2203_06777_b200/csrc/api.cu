// api.cu -- the C ABI of include/dwf.h: argument checking, geometry ownership, launch plumbing.
#include <stdarg.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "dwf_internal.cuh"

namespace dwf {

static thread_local char t_err[512] = "";
std::atomic<unsigned long long> g_launches{0};

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

// largest power-of-two exponent <= want that divides extent
static int fit_shift(int extent, int want)
{
    int s = 0;
    while (s < want && extent % (1 << (s + 1)) == 0) s++;
    return s;
}

// Tile table in launch order.  `raster` picks how the 4D grid of tiles is linearised; concurrently
// resident CTAs then cover a compact region so that halo re-reads hit in L2:
//   0: lexicographic, direction 0 fastest, time slowest
//   1: like 0, but direction 2 is split into two macro blocks swept one after the other
//   2: like 0, but direction 2 is split into four macro blocks
//   3: time fastest, then 0, 1, 2
static void build_tile_table(const Tiling &t, int raster, std::vector<int4> &tab)
{
    struct Digit { int dim, count; };
    std::vector<Digit> digits;   // fastest first
    auto split2 = [&](int nsplit) {
        int n2 = t.ntile[2];
        int outer = (n2 % nsplit == 0) ? nsplit : 1;
        digits = {{0, t.ntile[0]}, {1, t.ntile[1]}, {2, n2 / outer}, {3, t.ntile[3]}, {2, outer}};
    };
    switch (raster) {
    case 1: split2(2); break;
    case 2: split2(4); break;
    case 3: digits = {{3, t.ntile[3]}, {0, t.ntile[0]}, {1, t.ntile[1]}, {2, t.ntile[2]}}; break;
    default: digits = {{0, t.ntile[0]}, {1, t.ntile[1]}, {2, t.ntile[2]}, {3, t.ntile[3]}}; break;
    }
    tab.resize((size_t)t.ntiles);
    for (int id = 0; id < t.ntiles; id++) {
        int c[4] = {0, 0, 0, 0}, mult[4] = {1, 1, 1, 1};
        int r = id;
        for (const Digit &d : digits) {
            c[d.dim] += (r % d.count) * mult[d.dim];
            mult[d.dim] *= d.count;
            r /= d.count;
        }
        tab[(size_t)id] = make_int4(c[0] << t.sh[0], c[1] << t.sh[1], c[2] << t.sh[2], c[3] << t.sh[3]);
    }
}

static void make_tiling(const dwf_geometry *g, Tiling &t)
{
    const Lattice &lat = g->lat;
    const int ext[4] = {lat.Lh, lat.L[1], lat.L[2], lat.L[3]};
    int sites = 1;
    for (int d = 0; d < 4; d++) {
        t.sh[d] = fit_shift(ext[d], g->opt_tile[d]);
        t.ntile[d] = ext[d] >> t.sh[d];
        sites <<= t.sh[d];
    }
    // keep the CTA within 256 threads: shrink the tile from the slowest direction
    for (int d = 3; d >= 0 && sites > 256; d--)
        while (t.sh[d] > 0 && sites > 256) { t.sh[d]--; t.ntile[d] <<= 1; sites >>= 1; }
    int cpc = std::max(1, std::min(g->opt_cpc, 256 / sites));
    while (lat.Ls % cpc) cpc--;
    t.cpc = cpc;
    t.ncg = lat.Ls / cpc;
    t.threads = sites * cpc;
    t.ntiles = t.ntile[0] * t.ntile[1] * t.ntile[2] * t.ntile[3];
}

int rebuild_tilings(dwf_geometry *g)
{
    make_tiling(g, g->tiling_cb);
    std::vector<int4> tab;
    build_tile_table(g->tiling_cb, g->opt_raster, tab);
    if (g->tiles_cb) { cudaFree(g->tiles_cb); g->tiles_cb = nullptr; }
    DWF_CUDA_CHECK(cudaMalloc(&g->tiles_cb, tab.size() * sizeof(int4)));
    DWF_CUDA_CHECK(cudaMemcpy(g->tiles_cb, tab.data(), tab.size() * sizeof(int4), cudaMemcpyHostToDevice));

    if (g->tiles_staged) { cudaFree(g->tiles_staged); g->tiles_staged = nullptr; }
    plan_staged(g);
    if (g->staged.variant >= 0) {
        // [0, ntiles): the tiles of a half-field launch; [ntiles, 3 ntiles): the table of the full-field launch, every
        // tile twice with its output parity in .w (odd sites first, as two half launches would run)
        const size_t nt = (size_t)g->staged.ntiles;
        std::vector<int4> st(3 * nt);
        int raster = g->opt_raster_staged;
        if (raster < 0) {
            // auto: x1 fastest, x3 slowest, direction 2 split until a macro block has at most 96 tile
            // columns per x3 layer (C4: 128 -> 64, C5: 576 -> 72; measured optimum on both)
            const int n1 = g->lat.L[1] / g->staged.b[0], n2 = g->lat.L[2] / g->staged.b[1];
            raster = 0;
            while (raster < 9 && n1 * (n2 >> raster) > 96 && (n2 % (2 << raster)) == 0) raster++;
        }
        build_staged_tile_table(g, raster, st.data());
        for (size_t i = 0; i < nt; i++) {
            st[nt + i] = st[i];     st[nt + i].w = DWF_ODD;
            st[2 * nt + i] = st[i]; st[2 * nt + i].w = DWF_EVEN;
        }
        DWF_CUDA_CHECK(cudaMalloc(&g->tiles_staged, st.size() * sizeof(int4)));
        DWF_CUDA_CHECK(cudaMemcpy(g->tiles_staged, st.data(), st.size() * sizeof(int4), cudaMemcpyHostToDevice));
    }
    if (g->tiles_staged64) { cudaFree(g->tiles_staged64); g->tiles_staged64 = nullptr; }
    plan_staged64(g);
    if (g->staged64.variant >= 0) {
        std::vector<int4> st((size_t)g->staged64.ntiles);
        build_staged64_tile_table(g, st.data());
        DWF_CUDA_CHECK(cudaMalloc(&g->tiles_staged64, st.size() * sizeof(int4)));
        DWF_CUDA_CHECK(cudaMemcpy(g->tiles_staged64, st.data(), st.size() * sizeof(int4), cudaMemcpyHostToDevice));
    }
    return DWF_OK;
}

// ring of device buffers and copy streams for host transfers (dwf_internal.cuh: HostXfer)
static const size_t XFER_CHUNK = (size_t)32 << 20;

static int ensure_xfer(dwf_geometry *g)
{
    dwf_geometry::HostXfer &x = g->xfer;
    if (x.ready) return DWF_OK;
    x.chunk = XFER_CHUNK;
    for (int d = 0; d < 2; d++) {
        DWF_CUDA_CHECK(cudaStreamCreateWithFlags(&x.copy_stream[d], cudaStreamNonBlocking));
        for (int b = 0; b < 2; b++) {
            if (cudaMalloc(&x.buf[d][b], x.chunk) != cudaSuccess) {
                cudaGetLastError();
                set_error("cannot allocate %zu bytes of device staging", x.chunk);
                return DWF_ERR_ALLOC;
            }
            DWF_CUDA_CHECK(cudaEventCreateWithFlags(&x.filled[d][b], cudaEventDisableTiming));
            DWF_CUDA_CHECK(cudaEventCreateWithFlags(&x.drained[d][b], cudaEventDisableTiming));
        }
    }
    DWF_CUDA_CHECK(cudaStreamCreateWithFlags(&x.export_stream, cudaStreamNonBlocking));
    DWF_CUDA_CHECK(cudaEventCreateWithFlags(&x.export_begin, cudaEventDisableTiming));
    DWF_CUDA_CHECK(cudaEventCreateWithFlags(&x.export_done, cudaEventDisableTiming));
    x.ready = true;
    return DWF_OK;
}

static void destroy_xfer(dwf_geometry *g)
{
    dwf_geometry::HostXfer &x = g->xfer;
    for (int d = 0; d < 2; d++) {
        if (x.copy_stream[d]) { cudaStreamSynchronize(x.copy_stream[d]); cudaStreamDestroy(x.copy_stream[d]); }
        for (int b = 0; b < 2; b++) {
            cudaFree(x.buf[d][b]);
            if (x.filled[d][b]) cudaEventDestroy(x.filled[d][b]);
            if (x.drained[d][b]) cudaEventDestroy(x.drained[d][b]);
        }
    }
    if (x.export_stream) { cudaStreamSynchronize(x.export_stream); cudaStreamDestroy(x.export_stream); }
    if (x.export_begin) cudaEventDestroy(x.export_begin);
    if (x.export_done) cudaEventDestroy(x.export_done);
    memset(&x, 0, sizeof(x));
}

void wait_for_exports(const dwf_geometry *g, cudaStream_t st, const void *written, size_t bytes)
{
    const dwf_geometry::HostXfer &x = g->xfer;
    if (!x.ready || !x.export_pending) return;
    const char *w = static_cast<const char *>(written);
    if (w && (w + bytes <= x.export_ptr || x.export_ptr + x.export_bytes <= w)) return;      // disjoint
    cudaStreamWaitEvent(st, x.export_done, 0);
}

// canonical host array <-> device field in chunks of whole lattice lines (rows): a chunk of rows is a
// contiguous range of canonical sites.  IMPORT: H2D of chunk k+1 (copy stream) under the reorder of chunk k
// (caller's stream); export: reorder of chunk k+1 under the D2H of chunk k.
template <bool IMPORT>
static int host_transfer(dwf_geometry *g, const void *field_dev, void *field_dev_w, const void *host_src, void *host_dst, int parity,
                         cudaStream_t st)
{
    int rc = ensure_xfer(g);
    if (rc) return rc;
    dwf_geometry::HostXfer &x = g->xfer;
    const int d = IMPORT ? 0 : 1;
    const Lattice &lat = g->lat;
    const long long nrow = lat.Vh / lat.Lh;
    const size_t row_bytes = (size_t)(parity == DWF_FULL ? 2 : 1) * lat.Lh * lat.Ls * 24 * (size_t)g->prec;
    long long rows_per_chunk = (long long)(x.chunk / row_bytes);
    if (rows_per_chunk < 1) {          // a single lattice line larger than a ring buffer: grow the ring (rare: L0 * Ls * 96 B > 32 MB)
        destroy_xfer(g);
        rc = ensure_xfer(g);
        if (rc) return rc;
        for (int dd = 0; dd < 2; dd++)
            for (int b = 0; b < 2; b++) {
                cudaFree(x.buf[dd][b]);
                if (cudaMalloc(&x.buf[dd][b], row_bytes) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %zu bytes of device staging", row_bytes); return DWF_ERR_ALLOC; }
            }
        x.chunk = row_bytes;
        rows_per_chunk = 1;
    }
    cudaStream_t ks = st;           // stream of the reorder kernels
    if (IMPORT) {
        wait_for_exports(g, st, field_dev_w, dwf_field_bytes(g, parity));    // the import may overwrite a field that is still being exported
    } else {
        ks = x.export_stream;
        if (x.export_pending && x.export_ptr != field_dev) DWF_CUDA_CHECK(cudaStreamSynchronize(x.export_stream));   // one export tracked at a time
        x.export_ptr = static_cast<const char *>(field_dev);
        x.export_bytes = dwf_field_bytes(g, parity);
        DWF_CUDA_CHECK(cudaEventRecord(x.export_begin, st));
        DWF_CUDA_CHECK(cudaStreamWaitEvent(ks, x.export_begin, 0));
    }
    for (long long row0 = 0; row0 < nrow; row0 += rows_per_chunk) {
        const long long nr = (nrow - row0 < rows_per_chunk) ? nrow - row0 : rows_per_chunk;
        const int b = (int)(x.count[d]++ & 1);
        const size_t off = (size_t)row0 * row_bytes, bytes = (size_t)nr * row_bytes;
        if (IMPORT) {
            DWF_CUDA_CHECK(cudaStreamWaitEvent(x.copy_stream[0], x.drained[0][b], 0));
            DWF_CUDA_CHECK(cudaMemcpyAsync(x.buf[0][b], static_cast<const char *>(host_src) + off, bytes, cudaMemcpyHostToDevice, x.copy_stream[0]));
            DWF_CUDA_CHECK(cudaEventRecord(x.filled[0][b], x.copy_stream[0]));
            DWF_CUDA_CHECK(cudaStreamWaitEvent(st, x.filled[0][b], 0));
            if ((rc = launch_import(g, x.buf[0][b], parity, field_dev_w, st, row0, nr))) return rc;
            DWF_CUDA_CHECK(cudaEventRecord(x.drained[0][b], st));
        } else {
            DWF_CUDA_CHECK(cudaStreamWaitEvent(ks, x.drained[1][b], 0));
            if ((rc = launch_export(g, field_dev, parity, x.buf[1][b], ks, row0, nr))) return rc;
            DWF_CUDA_CHECK(cudaEventRecord(x.filled[1][b], ks));
            DWF_CUDA_CHECK(cudaStreamWaitEvent(x.copy_stream[1], x.filled[1][b], 0));
            DWF_CUDA_CHECK(cudaMemcpyAsync(static_cast<char *>(host_dst) + off, x.buf[1][b], bytes, cudaMemcpyDeviceToHost, x.copy_stream[1]));
            DWF_CUDA_CHECK(cudaEventRecord(x.drained[1][b], x.copy_stream[1]));
        }
    }
    if (!IMPORT) {
        DWF_CUDA_CHECK(cudaEventRecord(x.export_done, ks));
        x.export_pending = true;
    }
    if (!g->opt_async_host) {
        DWF_CUDA_CHECK(cudaStreamSynchronize(IMPORT ? st : x.copy_stream[1]));
        if (!IMPORT) x.export_pending = false;
    }
    return DWF_OK;
}

bool parity_ok(int p) { return p == DWF_FULL || p == DWF_EVEN || p == DWF_ODD; }
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

}  // namespace dwf

using namespace dwf;

extern "C" {

const char *dwf_error_string(int code)
{
    switch (code) {
    case DWF_OK: return "success";
    case DWF_ERR_INVALID_ARG: return "invalid argument";
    case DWF_ERR_BAD_GEOMETRY: return "bad geometry";
    case DWF_ERR_NO_GAUGE: return "gauge field not loaded";
    case DWF_ERR_CUDA: return "CUDA error";
    case DWF_ERR_ALLOC: return "allocation failed";
    case DWF_ERR_UNSUPPORTED: return "unsupported";
    }
    return "unknown error code";
}

const char *dwf_last_error(void) { return t_err; }

unsigned long long dwf_launch_count(void) { return g_launches.load(); }

int dwf_kernel_info(const dwf_geometry *g, char *buf, size_t n)
{
    if (!g || !buf || n == 0) { set_error("dwf_kernel_info: bad argument"); return DWF_ERR_INVALID_ARG; }
    const bool s32 = g->staged.variant >= 0 && g->opt_kernel != 1, s64 = g->staged64.variant >= 0 && g->opt_kernel != 1;
    if (s32)      snprintf(buf, n, "dhop_staged_kernel<%d,%d,%d,%d>", g->lat.Lh, g->staged.b[0], g->staged.b[1], g->staged.b[2]);
    else if (s64) snprintf(buf, n, "dhop_staged64%s_kernel<%d,%d,%d,%d>", g->staged64.kind == 2 ? "s" : (g->staged64.kind == 1 ? "t" : ""), g->lat.Lh,
                           g->staged64.b[0], g->staged64.b[1], g->staged64.b[2]);
    else          snprintf(buf, n, "dhop_direct_kernel<%s>", g->prec == DWF_F32 ? "float" : "double");
    return DWF_OK;
}

int dwf_create_geometry(const int dims[4], int Ls, int precision, int bc_time, int cuda_device, dwf_geometry **out)
{
    if (!dims || !out) { set_error("dwf_create_geometry: NULL argument"); return DWF_ERR_INVALID_ARG; }
    if (precision != DWF_F32 && precision != DWF_F64) { set_error("precision must be 4 or 8"); return DWF_ERR_UNSUPPORTED; }
    if (bc_time != DWF_PERIODIC && bc_time != DWF_ANTIPERIODIC_T && bc_time != DWF_OPEN_T) { set_error("bad bc_time"); return DWF_ERR_INVALID_ARG; }
    if (Ls < 1) { set_error("Ls must be >= 1"); return DWF_ERR_BAD_GEOMETRY; }
    long long V4 = 1;
    for (int d = 0; d < 4; d++) {
        if (dims[d] < 2 || (dims[d] & 1)) { set_error("extent %d is %d: must be even and >= 2", d, dims[d]); return DWF_ERR_BAD_GEOMETRY; }
        V4 *= dims[d];
        if (V4 > (1LL << 30)) { set_error("4D volume too large"); return DWF_ERR_BAD_GEOMETRY; }
    }
    if ((double)V4 * Ls * 12 >= 2147483647.0) { set_error("5D field exceeds 2^31 complex elements"); return DWF_ERR_BAD_GEOMETRY; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
        cudaGetLastError();
        set_error("CUDA device %d not available (%d devices)", cuda_device, ndev);
        return DWF_ERR_CUDA;
    }
    DeviceGuard guard(cuda_device);
    if (!guard.ok) { set_error("cannot select CUDA device %d", cuda_device); return DWF_ERR_CUDA; }

    dwf_geometry *g = new (std::nothrow) dwf_geometry();
    if (!g) return DWF_ERR_ALLOC;
    memset(g, 0, sizeof(*g));
    static std::atomic<unsigned long long> next_uid{1};
    g->uid = next_uid.fetch_add(1);
    for (int d = 0; d < 4; d++) g->lat.L[d] = dims[d];
    g->lat.Lh = dims[0] / 2;
    g->lat.Ls = Ls;
    g->lat.V4 = V4;
    g->lat.Vh = V4 / 2;
    g->prec = precision;
    g->bc_time = bc_time;
    g->device = cuda_device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) { delete g; set_error("cudaGetDeviceProperties failed"); return DWF_ERR_CUDA; }
    g->sm_count = prop.multiProcessorCount;
    g->opt_tile[0] = 4; g->opt_tile[1] = 2; g->opt_tile[2] = 1; g->opt_tile[3] = 1;
    g->opt_cpc = 1;
    g->opt_raster = 2;
    g->opt_raster_staged = -1;   // auto
    g->opt_variant = 0;
    g->opt_kernel = 0;
    g->opt_l2pol = 11222222;     // out, links evict_first; every input box evict_last (sweeps: least DRAM re-reads)
    g->opt_ssplit = 1;
    g->opt_zigzag = 1;
    g->opt_layered = 1;
    g->opt_full_launch = 1;

    g->gauge_bytes = (size_t)8 * 18 * (size_t)g->lat.Vh * (size_t)precision;
    g->reduce_blocks = g->sm_count * 32;
    bool ok = cudaMalloc(&g->gauge[0], g->gauge_bytes) == cudaSuccess &&
              cudaMalloc(&g->gauge[1], g->gauge_bytes) == cudaSuccess &&
              cudaMalloc(&g->tlink_top[0], (size_t)dims[1] * dims[2] * (dims[0] / 2) * 18 * (size_t)precision) == cudaSuccess &&
              cudaMalloc(&g->tlink_top[1], (size_t)dims[1] * dims[2] * (dims[0] / 2) * 18 * (size_t)precision) == cudaSuccess &&
              cudaMalloc(&g->partials, sizeof(double) * 2 * (size_t)g->reduce_blocks) == cudaSuccess &&
              cudaMalloc(&g->result_dev, sizeof(double) * 2) == cudaSuccess &&
              cudaHostAlloc(&g->mailbox_host, sizeof(double) * 4 * MAILBOX_SLOTS, cudaHostAllocMapped) == cudaSuccess &&
              cudaHostGetDevicePointer(&g->mailbox_dev, g->mailbox_host, 0) == cudaSuccess;
    if (ok) memset(g->mailbox_host, 0, sizeof(double) * 4 * MAILBOX_SLOTS);
    if (!ok || rebuild_tilings(g) != DWF_OK) {
        cudaGetLastError();
        if (ok == false) set_error("device allocation failed (gauge %zu bytes x 2)", g->gauge_bytes);
        dwf_destroy_geometry(g);
        return ok ? DWF_ERR_CUDA : DWF_ERR_ALLOC;
    }
    *out = g;
    return DWF_OK;
}

int dwf_destroy_geometry(dwf_geometry *g)
{
    if (!g) return DWF_OK;
    DeviceGuard guard(g->device);
    cudaFree(g->gauge[0]);
    cudaFree(g->gauge[1]);
    cudaFree(g->gauge12[0]);
    cudaFree(g->gauge12[1]);
    cudaFree(g->tlink_top[0]);
    cudaFree(g->tlink_top[1]);
    cudaFree(g->partials);
    cudaFree(g->result_dev);
    cudaFreeHost(g->mailbox_host);
    cudaFree(g->tiles_cb);
    cudaFree(g->tiles_staged);
    cudaFree(g->tiles_staged64);
    destroy_xfer(g);
    cudaGetLastError();
    delete g;
    return DWF_OK;
}

int dwf_set_option(dwf_geometry *g, const char *key, long long value)
{
    if (!g || !key) { set_error("dwf_set_option: NULL argument"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    int v = (int)value;
    if (!strcmp(key, "tile0") || !strcmp(key, "tile1") || !strcmp(key, "tile2") || !strcmp(key, "tile3")) {
        if (v < 0 || v > 8) { set_error("tile exponent out of range"); return DWF_ERR_INVALID_ARG; }
        g->opt_tile[key[4] - '0'] = v;
    } else if (!strcmp(key, "cpc")) {
        if (v < 1) { set_error("cpc must be >= 1"); return DWF_ERR_INVALID_ARG; }
        g->opt_cpc = v;
    } else if (!strcmp(key, "raster")) {
        g->opt_raster = v;
    } else if (!strcmp(key, "raster_staged")) {
        g->opt_raster_staged = v;
    } else if (!strcmp(key, "variant")) {
        g->opt_variant = v;          // 0: best staged tile, n > 0: n-th compiled staged variant only
    } else if (!strcmp(key, "l2pol")) {
        g->opt_l2pol = v;
        return DWF_OK;
    } else if (!strcmp(key, "zigzag")) {
        g->opt_zigzag = v != 0;
        return DWF_OK;
    } else if (!strcmp(key, "layered")) {
        g->opt_layered = v != 0;
        return DWF_OK;
    } else if (!strcmp(key, "ssplit")) {
        if (v < 1) { set_error("ssplit must be >= 1"); return DWF_ERR_INVALID_ARG; }
        g->opt_ssplit = v;
        return DWF_OK;
    } else if (!strcmp(key, "gauge12")) {
        if (v && g->prec != DWF_F32) { set_error("gauge12 needs an fp32 geometry"); return DWF_ERR_UNSUPPORTED; }
        g->opt_gauge12 = v != 0;
        if (g->opt_gauge12 && !g->gauge12[0]) g->gauge_loaded = false;        // takes effect at the next dwf_load_gauge
        return DWF_OK;
    } else if (!strcmp(key, "async_host")) {
        g->opt_async_host = v != 0;
        return DWF_OK;
    } else if (!strcmp(key, "full_launch")) {
        g->opt_full_launch = v != 0;
        return DWF_OK;
    } else if (!strcmp(key, "max_ctas")) {
        if (v < 0) { set_error("max_ctas must be >= 0"); return DWF_ERR_INVALID_ARG; }
        g->opt_max_ctas = (int)v;
        return DWF_OK;
    } else if (!strcmp(key, "kernel")) {
        if (v < 0 || v > 2) { set_error("kernel must be 0 (auto), 1 (direct) or 2 (staged)"); return DWF_ERR_INVALID_ARG; }
        g->opt_kernel = v;
        return DWF_OK;
    } else {
        set_error("unknown option '%s'", key);
        return DWF_ERR_UNSUPPORTED;
    }
    return rebuild_tilings(g);
}

size_t dwf_field_bytes(const dwf_geometry *g, int parity)
{
    if (!g || !parity_ok(parity)) return 0;
    const long long nsites = (parity == DWF_FULL) ? g->lat.V4 : g->lat.Vh;
    return (size_t)nsites * (size_t)g->lat.Ls * 24 * (size_t)g->prec;
}

int dwf_load_gauge(dwf_geometry *g, const void *U, int src_is_device, void *stream)
{
    if (!g || !U) { set_error("dwf_load_gauge: NULL argument"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t bytes = (size_t)g->lat.V4 * 72 * (size_t)g->prec;
    const void *src = U;
    void *tmp = nullptr;
    if (!src_is_device) {           // setup path: a temporary device copy of the canonical links, freed before returning
        if (cudaMalloc(&tmp, bytes) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate %zu bytes for the gauge upload", bytes); return DWF_ERR_ALLOC; }
        cudaError_t e = cudaMemcpyAsync(tmp, U, bytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { cudaFree(tmp); set_error("gauge upload failed: %s", cudaGetErrorString(e)); return DWF_ERR_CUDA; }
        src = tmp;
    }
    int rc = launch_pack_gauge(g, src, st);
    if (!rc) rc = launch_pack_tlinks(g, src, st);
    if (!rc && g->opt_gauge12) {
        // the compressed copy (two thirds of the bytes) next to the full one: only the plain staged fp32 Dhop reads it
        const size_t b12 = g->gauge_bytes / 3 * 2;
        for (int p = 0; p < 2 && !rc; p++)
            if (!g->gauge12[p] && cudaMalloc(&g->gauge12[p], b12) != cudaSuccess) { cudaGetLastError(); set_error("cannot allocate the 12-real gauge copy"); rc = DWF_ERR_ALLOC; }
        if (!rc) rc = launch_compress_gauge12(g, st);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    if (tmp) cudaFree(tmp);
    if (rc) return rc;
    if (e != cudaSuccess) { set_error("dwf_load_gauge failed: %s", cudaGetErrorString(e)); return DWF_ERR_CUDA; }
    g->gauge_loaded = true;
    return DWF_OK;
}

}  // extern "C"

// one half-Dhop: out (parity_out) = D in (opposite parity), or a x + b D in when axpy_x is given; picks
// the kernel.  Every kernel has the fused a x + b Dhop epilogue, x == out is allowed on all of them.
int dwf::half_dhop(const dwf_geometry *g, const void *in, void *out, int parity_out, cudaStream_t st, bool dagger,
                   const void *axpy_x, double a, double b, int nrhs)
{
    wait_for_exports(g, st, out, (size_t)nrhs * dwf_field_bytes(g, parity_out));
    const bool staged_any = g->staged.variant >= 0, staged64_ok = g->staged64.variant >= 0;
    const bool staged_ok = staged_any && (!axpy_x || staged_supports_axpy(g));
    // tiles whose x rows do not fit into shared memory next to the input slice (Lh = 32): staged Dhop, then
    // the elementwise pass -- possible whenever x is not the output buffer
    const bool staged_two_pass = staged_any && !staged_ok && axpy_x != out;
    if (g->opt_kernel == 2 && !staged_ok && !staged_two_pass && !staged64_ok) {
        set_error("the staged kernels do not support this geometry / precision");
        return DWF_ERR_UNSUPPORTED;
    }
    if (staged_ok && g->opt_kernel != 1)
        return launch_dhop_staged(g, in, out, parity_out, st, nullptr, nullptr, dagger, axpy_x, (float)a, (float)b, nrhs,
                                  g->opt_gauge12 && g->gauge12[0] && !dagger && !axpy_x);
    if (staged_two_pass && g->opt_kernel != 1) {
        int rc = launch_dhop_staged(g, in, out, parity_out, st, nullptr, nullptr, dagger, nullptr, 0.f, 0.f, nrhs);
        if (rc) return rc;
        return launch_axpby(g, axpy_x, out, a, b, (size_t)nrhs * dwf_field_bytes(g, parity_out) / (size_t)g->prec, st);
    }
    if (staged64_ok && g->opt_kernel != 1)
        return launch_dhop_staged64(g, in, out, parity_out, st, dagger, axpy_x, a, b, nullptr, nullptr, nrhs);
    // the direct kernel knows one field: one launch per right-hand side (the links are re-read)
    const size_t fb = dwf_field_bytes(g, parity_out);
    for (int r = 0; r < nrhs; r++) {
        const char *xi = axpy_x ? static_cast<const char *>(axpy_x) + r * fb : nullptr;
        int rc = launch_dhop_direct(g, static_cast<const char *>(in) + r * fb, static_cast<char *>(out) + r * fb, parity_out, st, dagger,
                                    xi, a, b);
        if (rc) return rc;
    }
    return DWF_OK;
}

extern "C" {

static int dhop_common(const dwf_geometry *g, const void *in, void *out, int parity_out, void *stream, const char *who,
                       bool dagger = false)
{
    if (!g || !in || !out) { set_error("%s: NULL argument", who); return DWF_ERR_INVALID_ARG; }
    if (in == out) { set_error("%s: in-place application is not defined (in == out)", who); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(out)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("%s: call dwf_load_gauge first", who); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (parity_out != DWF_FULL) return half_dhop(g, in, out, parity_out, st, dagger);
    // a full field is its even half field followed by its odd half field:
    // (Dhop psi)_odd = DhopOE psi_even, (Dhop psi)_even = DhopEO psi_odd
    // fp32 geometries with a staged variant: ONE launch whose tile table spans both parities
    if (!dagger && g->staged.variant >= 0 && g->opt_kernel != 1 && g->opt_full_launch && !(g->opt_gauge12 && g->gauge12[0])) {
        wait_for_exports(g, st, out, dwf_field_bytes(g, DWF_FULL));
        return launch_dhop_staged(g, in, out, DWF_FULL, st, nullptr, nullptr, false, nullptr, 0.f, 0.f, 1, false, true);
    }
    const size_t half = dwf_field_bytes(g, DWF_EVEN);
    const char *ie = static_cast<const char *>(in), *io = ie + half;
    char *oe = static_cast<char *>(out), *oo = oe + half;
    int rc = half_dhop(g, ie, oo, DWF_ODD, st, dagger);
    if (rc) return rc;
    return half_dhop(g, io, oe, DWF_EVEN, st, dagger);
}

int dwf_dhop(const dwf_geometry *g, const void *in_full, void *out_full, void *stream)
{
    return dhop_common(g, in_full, out_full, DWF_FULL, stream, "dwf_dhop");
}
int dwf_dhop_oe(const dwf_geometry *g, const void *in_even, void *out_odd, void *stream)
{
    return dhop_common(g, in_even, out_odd, DWF_ODD, stream, "dwf_dhop_oe");
}
int dwf_dhop_eo(const dwf_geometry *g, const void *in_odd, void *out_even, void *stream)
{
    return dhop_common(g, in_odd, out_even, DWF_EVEN, stream, "dwf_dhop_eo");
}
int dwf_dhop_dag(const dwf_geometry *g, const void *in_full, void *out_full, void *stream)
{
    return dhop_common(g, in_full, out_full, DWF_FULL, stream, "dwf_dhop_dag", true);
}
int dwf_dhop_oe_dag(const dwf_geometry *g, const void *in_even, void *out_odd, void *stream)
{
    return dhop_common(g, in_even, out_odd, DWF_ODD, stream, "dwf_dhop_oe_dag", true);
}
int dwf_dhop_eo_dag(const dwf_geometry *g, const void *in_odd, void *out_even, void *stream)
{
    return dhop_common(g, in_odd, out_even, DWF_EVEN, stream, "dwf_dhop_eo_dag", true);
}

// nrhs right-hand sides in one launch, one gauge load for all of them
static int dhop_mrhs_common(const dwf_geometry *g, const void *in, void *out, int parity_out, int nrhs, int dagger, void *stream,
                            const char *who)
{
    if (!g || !in || !out || nrhs < 1) { set_error("%s: NULL argument or nrhs < 1", who); return DWF_ERR_INVALID_ARG; }
    if (in == out) { set_error("%s: in-place application is not defined (in == out)", who); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(out)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    if ((double)g->lat.L[3] * g->lat.Ls * nrhs >= 2147483647.0) { set_error("%s: L3 * Ls * nrhs exceeds 2^31", who); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("%s: call dwf_load_gauge first", who); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    return half_dhop(g, in, out, parity_out, static_cast<cudaStream_t>(stream), dagger != 0, nullptr, 0.0, 0.0, nrhs);
}
int dwf_dhop_oe_mrhs(const dwf_geometry *g, const void *in_even, void *out_odd, int nrhs, int dagger, void *stream)
{
    return dhop_mrhs_common(g, in_even, out_odd, DWF_ODD, nrhs, dagger, stream, "dwf_dhop_oe_mrhs");
}
int dwf_dhop_eo_mrhs(const dwf_geometry *g, const void *in_odd, void *out_even, int nrhs, int dagger, void *stream)
{
    return dhop_mrhs_common(g, in_odd, out_even, DWF_EVEN, nrhs, dagger, stream, "dwf_dhop_eo_mrhs");
}

}  // extern "C"

// Waits for the reduction last enqueued on `st` and returns its n values.  The final-sum kernel
// writes them into mapped host memory followed by its sequence number, so the host polls that
// word instead of paying a device-to-host copy plus a stream synchronise; cudaStreamQuery is
// consulted now and then so that a failed launch surfaces as an error instead of a hang.  When the
// sequence number is visible every earlier operation of the stream has completed (in-order stream).
int dwf::fetch_reduction(const dwf_geometry *g, cudaStream_t st, int n, double *out, unsigned long long ticket)
{
    const unsigned long long want = ticket ? ticket : g->mailbox_seq;
    if (want == 0 || want > g->mailbox_seq || g->mailbox_seq - want >= MAILBOX_SLOTS) {
        set_error("reduction %llu is not pending (last issued %llu, at most %llu results are kept)", want, g->mailbox_seq, MAILBOX_SLOTS);
        return DWF_ERR_INVALID_ARG;
    }
    const double *slot = g->mailbox_host + 4 * (want % MAILBOX_SLOTS);
    volatile unsigned long long *seq = reinterpret_cast<volatile unsigned long long *>(const_cast<double *>(slot) + 2);
    for (unsigned long long spins = 1; *seq != want; spins++) {
        if ((spins & 0x3fff) == 0) {
            cudaError_t e = cudaStreamQuery(st);
            if (e == cudaSuccess) break;               // stream drained: the values are there
            if (e != cudaErrorNotReady) { set_error("reduction failed: %s", cudaGetErrorString(e)); return DWF_ERR_CUDA; }
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    if (*seq != want) {
        DWF_CUDA_CHECK(cudaStreamSynchronize(st));
        if (*seq != want) {        // the stream drained without the final-sum kernel of this call having run
            set_error("reduction result never arrived (sequence %llu, expected %llu)", *seq, want);
            return DWF_ERR_CUDA;
        }
    }
    for (int i = 0; i < n; i++) out[i] = const_cast<const volatile double *>(slot)[i];
    return DWF_OK;
}

extern "C" {

// out = D in on half fields and *result_host = norm2(out): the reduction runs in the epilogue of the
// Dhop kernel (staged path) or as a second pass over `out` (direct path)
static int dhop_norm2_common(const dwf_geometry *g, const void *in, void *out, int parity_out, double *result_host,
                             void *stream, const char *who, unsigned long long *ticket = nullptr)
{
    if (!g || !in || !out || (!result_host && !ticket)) { set_error("%s: NULL argument", who); return DWF_ERR_INVALID_ARG; }
    if (in == out) { set_error("%s: in-place application is not defined (in == out)", who); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(out)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("%s: call dwf_load_gauge first", who); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    wait_for_exports(g, st, out, dwf_field_bytes(g, parity_out));
    const bool staged_ok = g->staged.variant >= 0;
    if (g->opt_kernel == 2 && !staged_ok && g->staged64.variant < 0) {
        set_error("the staged kernel does not support this geometry / precision");
        return DWF_ERR_UNSUPPORTED;
    }
    int rc;
    if (staged_ok && g->opt_kernel != 1) {
        int nblocks = 0;
        rc = launch_dhop_staged(g, in, out, parity_out, st, g->partials, &nblocks);
        if (rc) return rc;
        rc = launch_final_sum(g, nblocks, st);
    } else if (g->staged64.variant >= 0 && g->opt_kernel != 1) {
        int nblocks = 0;
        rc = launch_dhop_staged64(g, in, out, parity_out, st, false, nullptr, 0.0, 0.0, g->partials, &nblocks);
        if (rc) return rc;
        rc = launch_final_sum(g, nblocks, st);
    } else {
        rc = half_dhop(g, in, out, parity_out, st);
        if (rc) return rc;
        rc = launch_norm2(g, out, dwf_field_bytes(g, parity_out) / (size_t)g->prec, st);
    }
    if (rc) return rc;
    if (ticket) { *ticket = g->mailbox_seq; return DWF_OK; }       // asynchronous form: the caller collects the value later
    return fetch_reduction(g, st, 1, result_host);
}

int dwf_dhop_oe_norm2_async(const dwf_geometry *g, const void *in_even, void *out_odd, unsigned long long *ticket, void *stream)
{
    return dhop_norm2_common(g, in_even, out_odd, DWF_ODD, nullptr, stream, "dwf_dhop_oe_norm2_async", ticket);
}
int dwf_dhop_eo_norm2_async(const dwf_geometry *g, const void *in_odd, void *out_even, unsigned long long *ticket, void *stream)
{
    return dhop_norm2_common(g, in_odd, out_even, DWF_EVEN, nullptr, stream, "dwf_dhop_eo_norm2_async", ticket);
}
int dwf_reduction_wait(const dwf_geometry *g, unsigned long long ticket, double *result_host, void *stream)
{
    if (!g || !result_host || !ticket) { set_error("dwf_reduction_wait: bad argument"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    return fetch_reduction(g, static_cast<cudaStream_t>(stream), 1, result_host, ticket);
}

int dwf_dhop_oe_norm2(const dwf_geometry *g, const void *in_even, void *out_odd, double *result_host, void *stream)
{
    return dhop_norm2_common(g, in_even, out_odd, DWF_ODD, result_host, stream, "dwf_dhop_oe_norm2");
}
int dwf_dhop_eo_norm2(const dwf_geometry *g, const void *in_odd, void *out_even, double *result_host, void *stream)
{
    return dhop_norm2_common(g, in_odd, out_even, DWF_EVEN, result_host, stream, "dwf_dhop_eo_norm2");
}

// out = a x + b (D in) on half fields: one pass in the staged kernel, Dhop then axpby otherwise
static int dhop_axpy_common(const dwf_geometry *g, const void *in, const void *x, double a, double b, void *out,
                            int parity_out, void *stream, const char *who)
{
    if (!g || !in || !x || !out) { set_error("%s: NULL argument", who); return DWF_ERR_INVALID_ARG; }
    if (in == out || in == x) { set_error("%s: `in` must differ from `x` and `out` (x == out is allowed)", who); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(in) || !aligned16(out) || !aligned16(x)) { set_error("%s: field pointers must be 16-byte aligned", who); return DWF_ERR_INVALID_ARG; }
    if (!g->gauge_loaded) { set_error("%s: call dwf_load_gauge first", who); return DWF_ERR_NO_GAUGE; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return half_dhop(g, in, out, parity_out, st, false, x, a, b);
}

int dwf_dhop_oe_axpy(const dwf_geometry *g, const void *in_even, const void *x_odd, double a, double b, void *out_odd, void *stream)
{
    return dhop_axpy_common(g, in_even, x_odd, a, b, out_odd, DWF_ODD, stream, "dwf_dhop_oe_axpy");
}
int dwf_dhop_eo_axpy(const dwf_geometry *g, const void *in_odd, const void *x_even, double a, double b, void *out_even, void *stream)
{
    return dhop_axpy_common(g, in_odd, x_even, a, b, out_even, DWF_EVEN, stream, "dwf_dhop_eo_axpy");
}

int dwf_norm2(const dwf_geometry *g, const void *field, int parity, double *result_host, void *stream)
{
    if (!g || !field || !result_host || !parity_ok(parity)) { set_error("dwf_norm2: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(field)) { set_error("dwf_norm2: field must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = launch_norm2(g, field, dwf_field_bytes(g, parity) / (size_t)g->prec, st);
    if (rc) return rc;
    return fetch_reduction(g, st, 1, result_host);
}

int dwf_inner_product(const dwf_geometry *g, const void *a, const void *b, int parity, double result_host[2], void *stream)
{
    if (!g || !a || !b || !result_host || !parity_ok(parity)) { set_error("dwf_inner_product: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(a) || !aligned16(b)) { set_error("dwf_inner_product: fields must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = launch_inner(g, a, b, dwf_field_bytes(g, parity) / (size_t)g->prec / 2, st);
    if (rc) return rc;
    return fetch_reduction(g, st, 2, result_host);
}

int dwf_import_spinor(const dwf_geometry *g, const void *canonical, int src_is_device, int parity, void *field_dev, void *stream)
{
    if (!g || !canonical || !field_dev || !parity_ok(parity)) { set_error("dwf_import_spinor: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(field_dev) || (src_is_device && !aligned16(canonical))) { set_error("dwf_import_spinor: device pointers must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    if (canonical == field_dev) { set_error("dwf_import_spinor: in-place conversion not supported"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (!src_is_device) return host_transfer<true>(const_cast<dwf_geometry *>(g), nullptr, field_dev, canonical, nullptr, parity, st);
    return launch_import(g, canonical, parity, field_dev, st);
}

int dwf_export_spinor(const dwf_geometry *g, const void *field_dev, int parity, void *canonical, int dst_is_device, void *stream)
{
    if (!g || !canonical || !field_dev || !parity_ok(parity)) { set_error("dwf_export_spinor: bad argument"); return DWF_ERR_INVALID_ARG; }
    if (!aligned16(field_dev) || (dst_is_device && !aligned16(canonical))) { set_error("dwf_export_spinor: device pointers must be 16-byte aligned"); return DWF_ERR_INVALID_ARG; }
    if (canonical == field_dev) { set_error("dwf_export_spinor: in-place conversion not supported"); return DWF_ERR_INVALID_ARG; }
    DeviceGuard guard(g->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (dst_is_device) return launch_export(g, field_dev, parity, canonical, st);
    return host_transfer<false>(const_cast<dwf_geometry *>(g), field_dev, nullptr, nullptr, canonical, parity, st);
}

int dwf_host_wait(const dwf_geometry *g)
{
    if (!g) { set_error("dwf_host_wait: NULL argument"); return DWF_ERR_INVALID_ARG; }
    if (!g->xfer.ready) return DWF_OK;
    DeviceGuard guard(g->device);
    DWF_CUDA_CHECK(cudaStreamSynchronize(g->xfer.copy_stream[0]));
    DWF_CUDA_CHECK(cudaStreamSynchronize(g->xfer.copy_stream[1]));
    const_cast<dwf_geometry *>(g)->xfer.export_pending = false;
    return DWF_OK;
}

}  // extern "C"

/*
 * dwf.h -- C ABI of libdwf: the Domain Wall Fermion hopping term Dhop on one B200.
 *
 * The operation (BASELINE.json north_star; the paper names it "the Domain Wall Fermion
 * operator", section 1, "node local 'Wilson' matrix", L223 section 4, "main kernel
 * DWF code", L254 Fig.6, and never prints it -- SURVEY.md 8(c) reading #1):
 *
 *   Dhop psi(x,s) = sum_{mu=0..3} [ (1 - gamma_mu) U_mu(x)        psi(x+mu,s)
 *                                 + (1 + gamma_mu) U_mu^dag(x-mu) psi(x-mu,s) ]
 *
 * x runs over a 4D lattice L0 x L1 x L2 x L3 (mu = 0,1,2,3 = x,y,z,t; time is the LAST extent),
 * s = 0..Ls-1 is a spectator index, psi(x,s) has 4 spin x 3 colour complex components, U_mu(x)
 * is a 3x3 complex matrix acting on colour.  DeGrand-Rossi gamma basis.  Boundaries are
 * periodic; with DWF_ANTIPERIODIC_T a hop that wraps around the time direction gets a factor -1.
 * No prefactor, no mass term, no fifth-dimension hopping.  1320 flop per output 5D site.
 *
 * Everything is extern "C", plain pointers and sizes.  Every function returns a DWF_* status
 * (0 = success); on error no output is written; nothing aborts or throws.  dwf_last_error()
 * returns a thread-local detail string for the last failing call of the calling thread.
 *
 * CANONICAL (interchange) layouts, reals of the geometry's precision, C order:
 *   site     x = x0 + L0*(x1 + L1*(x2 + L2*x3))
 *   parity   p(x) = (x0+x1+x2+x3) & 1  (s is not included)
 *   gauge    [x][mu][a][b][reim]            U_mu(x)_{ab}: row a, column b, (U psi)_a = sum_b U_ab psi_b
 *   spinor   [site][s][spin][colour][reim]  site = x (full field), or x>>1 for a half field that
 *                                           holds the sites of one parity in increasing x
 *
 * DEVICE field layout (what `field`, `in`, `out` pointers below hold; produced only by
 * dwf_import_spinor, read back only by dwf_export_spinor; size dwf_field_bytes):
 *   half field   pair[s][row][k/2][h][k&1]: row = x1 + L1*(x2 + L2*x3) (a lattice line along x0),
 *                h = x0>>1 (cb site x>>1 = row*Lh + h), 12 slots k of two reals per site, slots
 *                2j and 2j+1 adjacent (one 128-bit vector in fp32).
 *                fp64: complex[s][row][k][h] instead, k = spin*3 + colour: one plane per component,
 *                a site's complex number (re, im) is one 128-bit word.
 *                fp32: slot k = 4*colour + t = one real part of a pair of spins, t = 0 (re of
 *                spins 0,1), 1 (im of 0,1), 2 (re of 2,3), 3 (im of 2,3).
 *   full field   the even half field followed by the odd half field
 *   "SoA complex components, site-fastest" (north_star subsystem 1).  s is the SLOWEST index: the
 *   fast kernel keeps the 8 links of a 4D site in registers and walks through all Ls slices, so
 *   each link is loaded once per 4D site and every slice is a dense 4D tensor that TMA can tile
 *   (DESIGN.md "Data layout" says why this replaces the "Ls innermost" of north_star).
 * Device pointers must be 16-byte aligned and live on the geometry's device.
 * `stream` is a cudaStream_t passed as void* (NULL = the default stream).
 */
#ifndef DWF_H
#define DWF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define DWF_API __attribute__((visibility("default")))
#else
#define DWF_API
#endif

typedef struct dwf_geometry dwf_geometry;   /* opaque, library-owned */

enum { DWF_OK = 0, DWF_ERR_INVALID_ARG = 1, DWF_ERR_BAD_GEOMETRY = 2, DWF_ERR_NO_GAUGE = 3,
       DWF_ERR_CUDA = 4, DWF_ERR_ALLOC = 5, DWF_ERR_UNSUPPORTED = 6 };
enum { DWF_F32 = 4, DWF_F64 = 8 };                   /* precision = bytes per real            */
enum { DWF_PERIODIC = 0, DWF_ANTIPERIODIC_T = 1,     /* time = dims[3]                        */
       DWF_OPEN_T = 2 };                             /* hops that would wrap in time contribute nothing: one time slab of a
                                                        domain-decomposed lattice (dwf_face_pack_t / dwf_face_apply_t)     */
enum { DWF_FULL = -1, DWF_EVEN = 0, DWF_ODD = 1 };   /* parity = (x0+x1+x2+x3) & 1            */

/* Create a geometry: lattice extents dims[4] (each even and >= 2), fifth-dimension extent Ls >= 1,
 * precision DWF_F32 / DWF_F64 (storage AND arithmetic; no mixed precision), bc_time, CUDA device
 * ordinal.  Allocates the device gauge storage and reduction scratch (owned by the geometry).
 * Errors: INVALID_ARG (NULL), BAD_GEOMETRY (odd or < 2 extent, Ls < 1, field too large: a full 5D field is
 * limited to 2^31 - 1 complex numbers, i.e. V4 * Ls * 12 < 2^31 -- C5 has 1.5e9 -- and V4 to 2^30 sites),
 * UNSUPPORTED (precision), CUDA / ALLOC.
 *
 * CONCURRENCY.  dwf_dhop, dwf_dhop_oe/eo, their _dag, _axpy, _mrhs and _f16 forms, dwf_to_f16 / dwf_from_f16, dwf_mooee,
 * dwf_mooee_inv, dwf_ddwf, dwf_schur and dwf_axpby only read the geometry: they may be called concurrently on different streams.
 * Calls that use the geometry's scratch -- dwf_norm2, dwf_inner_product, dwf_dhop_oe_norm2 / _eo_norm2 and their _async
 * forms, dwf_reduction_wait, dwf_cg_schur (reduction partials and the result mailbox), dwf_import_spinor / dwf_export_spinor with HOST
 * arrays and dwf_host_wait (the transfer ring) -- must be serialised by the caller per geometry (one at a
 * time; they may overlap with the read-only calls).  dwf_load_gauge, dwf_set_option and dwf_destroy_geometry
 * must not race with anything on the same geometry. */
DWF_API int dwf_create_geometry(const int dims[4], int Ls, int precision, int bc_time, int cuda_device,
                        dwf_geometry **out);

/* Free everything the geometry owns.  Must not race with any other call on g. */
DWF_API int dwf_destroy_geometry(dwf_geometry *g);

/* Load (or replace) the gauge field from the canonical layout; src_is_device says where
 * U_canonical lives (host memory need not be pinned).  Builds the device copies: for every output
 * site the 8 links it needs, U_mu(x) and the pre-daggered U_mu^dag(x-mu), with the antiperiodic
 * sign folded in.  Synchronises `stream` before returning: the caller may free U_canonical. */
DWF_API int dwf_load_gauge(dwf_geometry *g, const void *U_canonical, int src_is_device, void *stream);

/* out = Dhop in on full fields (device layout).  Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL, in == out, misaligned), NO_GAUGE, CUDA.  Partial overlap of in and
 * out is undefined. */
DWF_API int dwf_dhop(const dwf_geometry *g, const void *in_full, void *out_full, void *stream);

/* Checkerboarded variants, first letter = output parity (SURVEY.md 8(c) reading #6):
 * DhopOE: even half field in -> odd half field out;  DhopEO: odd in -> even out.
 * (Dhop psi)_odd = DhopOE psi_even, (Dhop psi)_even = DhopEO psi_odd.  Asynchronous. */
DWF_API int dwf_dhop_oe(const dwf_geometry *g, const void *in_even, void *out_odd, void *stream);
DWF_API int dwf_dhop_eo(const dwf_geometry *g, const void *in_odd, void *out_even, void *stream);

/* The adjoint operator (the first NEXT row; needed for CG on the normal equations):
 *   Dhop^dag psi(x,s) = sum_mu [ (1+gamma_mu) U_mu(x) psi(x+mu,s) + (1-gamma_mu) U_mu^dag(x-mu) psi(x-mu,s) ]
 * = gamma5 Dhop gamma5 (the hop matrices change places under the adjoint, gamma_mu is Hermitian, so
 * only the projectors swap; PAPER.md never writes the operator, BASELINE.json north_star does).
 * Same layouts, parities (first letter = output parity), errors and asynchrony as the calls above. */
DWF_API int dwf_dhop_dag(const dwf_geometry *g, const void *in_full, void *out_full, void *stream);
DWF_API int dwf_dhop_oe_dag(const dwf_geometry *g, const void *in_even, void *out_odd, void *stream);
DWF_API int dwf_dhop_eo_dag(const dwf_geometry *g, const void *in_odd, void *out_even, void *stream);

/* The Wilson-matrix fusion of SURVEY.md 8(f1):  out = a x + b (DhopOE in)   resp.   a x + b (DhopEO in),
 * x and out half fields of the OUTPUT parity.  With a = 4 + m, b = -1/2 this is one half of the
 * even/odd Wilson matrix M = (4 + m) - Dhop/2, with a = 1 one half of its Schur complement.  Every
 * kernel combines in its store epilogue (one pass; the fast fp32 kernel stages x by TMA next to the input
 * slice); x == out is allowed.  a, b are rounded to the geometry's precision.  `in` must differ
 * from x and out.  Asynchronous on `stream`.  Errors as dwf_dhop_oe. */
DWF_API int dwf_dhop_oe_axpy(const dwf_geometry *g, const void *in_even, const void *x_odd, double a, double b,
                     void *out_odd, void *stream);
DWF_API int dwf_dhop_eo_axpy(const dwf_geometry *g, const void *in_odd, const void *x_even, double a, double b,
                     void *out_even, void *stream);

/* Multiple right-hand sides sharing one gauge load (not in PAPER.md).  `in` and `out` hold
 * nrhs half fields of the device layout one after the other (nrhs * dwf_field_bytes(g, parity) bytes each);
 * out_r = DhopOE in_r (dagger != 0: the adjoint) for every r, identical bit for bit to nrhs separate calls.
 * Dhop does not couple the slices s, so to the staged kernels the nrhs fields are ONE field of nrhs * Ls
 * slices: a thread loads its 8 links once and walks all of them.  Minimal-traffic model: w (48 + 144 / (Ls
 * nrhs)) bytes per output 5D site instead of w (48 + 144 / Ls).  The general (direct) kernel runs one launch
 * per right-hand side.  Asynchronous.  Errors as dwf_dhop_oe; INVALID_ARG for nrhs < 1 or L3 Ls nrhs >= 2^31. */
DWF_API int dwf_dhop_oe_mrhs(const dwf_geometry *g, const void *in_even, void *out_odd, int nrhs, int dagger, void *stream);
DWF_API int dwf_dhop_eo_mrhs(const dwf_geometry *g, const void *in_odd, void *out_even, int nrhs, int dagger, void *stream);

/* ---- Domain decomposition along time ("near perfect overlap of communication
 * and computation", L250 "face assembly"; reading #26).  A rank owns a slab of dims[3] time layers and
 * creates its geometry with DWF_OPEN_T; dwf_dhop_oe / _eo (and their _dag forms) then compute everything but the
 * two face terms.  Per half-Dhop (in of parity q = 1 - p, out of parity p):
 *   1. dwf_face_pack_t(g, in, q, dagger, send_down, send_up): projected half spinors (12 reals per face site and
 *      slice, dwf_face_bytes(g) bytes per buffer) of the slab's first layer for the LOWER neighbour (send_down) and of
 *      its last layer, already multiplied by U_t^dag, for the UPPER neighbour (send_up);
 *   2. the exchange (outside this library: NCCL send / recv, a peer copy, or a plain copy when the rank is its own
 *      neighbour), overlapped with 3. the bulk half-Dhop on `stream`;
 *   4. dwf_face_apply_t(g, recv_lo, recv_hi, sign_lo, sign_hi, out, p, dagger): recv_lo = the lower neighbour's
 *      send_up, recv_hi = the upper neighbour's send_down; adds sign_lo (1 + gamma_t) [recv_lo] to the first layer
 *      and sign_hi (1 - gamma_t) U_t(x) [recv_hi] to the last layer of out (sign = -1 on the face that crosses a
 *      global antiperiodic boundary, else +1).
 * The assembled result equals the Dhop of the whole lattice.  All asynchronous on `stream`; device pointers,
 * 16-byte aligned.  Errors: INVALID_ARG, NO_GAUGE, CUDA. */
DWF_API size_t dwf_face_bytes(const dwf_geometry *g);
DWF_API int dwf_face_pack_t(const dwf_geometry *g, const void *in, int parity_in, int dagger, void *send_down, void *send_up,
                            void *stream);
DWF_API int dwf_face_apply_t(const dwf_geometry *g, const void *recv_lo, const void *recv_hi, double sign_lo, double sign_hi,
                             void *out, int parity_out, int dagger, void *stream);

/* *result_host = sum over all reals of |field|^2, accumulated in fp64 in a fixed order
 * (deterministic).  parity = DWF_FULL for a full field, DWF_EVEN / DWF_ODD for a half field.
 * Synchronises `stream`. */
DWF_API int dwf_norm2(const dwf_geometry *g, const void *field, int parity, double *result_host,
              void *stream);

/* ---- fp16 STORAGE of spinor fields, fp32 arithmetic (third variant; not in PAPER.md).  A field in fp16
 * storage is the fp32 DEVICE layout element by element with IEEE binary16 reals: dwf_field_bytes(g, parity) / 2 bytes, a
 * device pointer, 16-byte aligned, owned by the caller.  The links stay fp32.  fp32 geometries only (UNSUPPORTED otherwise).
 * dwf_to_f16: field_f16 = round-to-nearest-even(field_f32); dwf_from_f16: exact widening.  Asynchronous on `stream`.
 * dwf_dhop_oe_f16 / dwf_dhop_eo_f16: out = round_f16( Dhop( widen(in) ) ): every input real is widened to fp32 after the
 * shared-memory load, projection, SU(3) products and the sum over the 8 legs run in fp32 exactly as in dwf_dhop_oe / _eo,
 * and the result is rounded ONCE (nearest even) in the store.  Traffic model: 96 + 576/Ls bytes per 5D output site (132 at
 * Ls = 16 against 228 in fp32).  Needs a staged variant whose fp16 rows stay 128-byte aligned: L0 a
 * multiple of 16 (UNSUPPORTED otherwise; there is no fp16 path through the general kernel).  Overflow is the caller's
 * concern (|values| <= 65504).  Errors: INVALID_ARG (NULL, alignment, in == out), NO_GAUGE, UNSUPPORTED, CUDA. */
DWF_API int dwf_to_f16(const dwf_geometry *g, const void *field_f32, int parity, void *field_f16, void *stream);
DWF_API int dwf_from_f16(const dwf_geometry *g, const void *field_f16, int parity, void *field_f32, void *stream);
DWF_API int dwf_dhop_oe_f16(const dwf_geometry *g, const void *in_even_f16, void *out_odd_f16, void *stream);
DWF_API int dwf_dhop_eo_f16(const dwf_geometry *g, const void *in_odd_f16, void *out_even_f16, void *stream);

/* norm2 WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): no geometry is needed, and the per-CTA partial sums live in a file-scope __device__
 * array of the library (512.25 KB, held by every GPU that loads the library until the process exits) instead of the
 * scratch a geometry allocates.  *result_dev = sum over the n_reals reals at x_dev of x^2, accumulated in fp64 in a
 * fixed order (deterministic; it differs from dwf_norm2 of the same buffer only in summation order, relative
 * difference <= 1e-12).  x_dev: device pointer on cuda_device, 16-byte aligned, n_reals values of `precision`
 * (DWF_F32 / DWF_F64), any buffer (a field in device layout, or anything else); result_dev: device pointer to ONE
 * double, 8-byte aligned, owned by the caller, written asynchronously on `stream` (the call does not synchronise
 * and copies nothing to the host).  The call issues one memset of the arrival counter and one kernel on `stream`
 * and calls no cudaMalloc / cudaFree or allocating routine; the first call on a device looks the array's address
 * up (cudaGetSymbolAddress), so make one call outside a capture first.
 * LIMIT: n_reals * precision <= DWF_NORM2_STATIC_MAX_BYTES (2 GiB: 2^29 fp32 or 2^28 fp64 values; a C4 half
 * field is 0.8 / 1.6 GB); larger buffers are rejected with INVALID_ARG and a message naming the limit.
 * SHARING: every call on a device uses the same array.  Calls that may overlap on the GPU (different streams,
 * parallel graph branches, several host threads) race on it: the caller serialises them.
 * Errors: INVALID_ARG (NULL, alignment, size, device ordinal), UNSUPPORTED (precision), CUDA. */
#define DWF_NORM2_STATIC_MAX_BYTES ((size_t)1 << 31)
DWF_API int dwf_norm2_static(const void *x_dev, size_t n_reals, int precision, int cuda_device, double *result_dev,
                             void *stream);

/* DhopOE / DhopEO fused with the norm2 of their result (SURVEY.md 8(a) rows a6 + a7 in one pass):
 * out = D in and *result_host = sum |out|^2, fp64 accumulation in a fixed order (deterministic
 * for a given geometry and option set; it differs from dwf_norm2(out) only in summation order,
 * relative difference <= 1e-12).  The fast fp32 kernel accumulates in its epilogue, so the
 * output field is not read again; other geometries run the two passes.  Arguments and errors
 * as dwf_dhop_oe / dwf_dhop_eo; synchronises `stream` like dwf_norm2. */
DWF_API int dwf_dhop_oe_norm2(const dwf_geometry *g, const void *in_even, void *out_odd, double *result_host, void *stream);
DWF_API int dwf_dhop_eo_norm2(const dwf_geometry *g, const void *in_odd, void *out_even, double *result_host, void *stream);

/* The same two calls WITHOUT the wait: the kernels are enqueued on `stream`, *ticket names the reduction, and the call
 * returns at once; dwf_reduction_wait(g, ticket, &value, stream) later waits for that reduction (same `stream`) and
 * returns its value -- so that a caller can enqueue the next step's kernels before it reads this step's norm and the GPU
 * never idles on the host (`bench.py` does).  The library keeps the results of the last 8 reductions of a geometry
 * (every dwf_norm2, dwf_inner_product, dwf_dhop_*_norm2[_async] and every reduction inside dwf_cg_schur counts): waiting
 * for an older ticket is INVALID_ARG.  The serialisation rule of the geometry's scratch (above) applies unchanged: all of
 * these calls on one geometry go to ONE stream, one host thread at a time. */
DWF_API int dwf_dhop_oe_norm2_async(const dwf_geometry *g, const void *in_even, void *out_odd, unsigned long long *ticket, void *stream);
DWF_API int dwf_dhop_eo_norm2_async(const dwf_geometry *g, const void *in_odd, void *out_even, unsigned long long *ticket, void *stream);
DWF_API int dwf_reduction_wait(const dwf_geometry *g, unsigned long long ticket, double *result_host, void *stream);

/* result_host[0..1] = (re, im) of sum conj(a) b.  Same rules as dwf_norm2. */
DWF_API int dwf_inner_product(const dwf_geometry *g, const void *a, const void *b, int parity,
                      double result_host[2], void *stream);

/* ---- The rest of the red-black domain-wall operator (section 4: "all
 * kernels involved in the DWF Dirac operator", L250 Fig.5, L254 Fig.6 -- named, never printed).  The
 * definition is the standard Shamir domain-wall matrix (reading #22), with domain-wall
 * height M5 and fermion mass `mass`:
 *
 *   (M psi)(x,s) = (5 - M5) psi(x,s) - 1/2 (Dhop psi)(x,s) - P_- psi(x,s+1) - P_+ psi(x,s-1),
 *   P_+- = (1 +- gamma5)/2, gamma5 = diag(+1,+1,-1,-1),  psi(x,Ls) = -mass psi(x,0),  psi(x,-1) = -mass psi(x,Ls-1).
 *
 * "Mooee" is M without the Dhop term: diagonal in the 4D site, it couples the slices s of one site.
 * With the 4D checkerboard, M = [Mee Meo; Moe Moo] with Mee = Moo = Mooee, Meo = -1/2 DhopEO,
 * Moe = -1/2 DhopOE.  `dagger` != 0 selects the adjoint of the operator everywhere below.
 * All fields are in the device layout; all calls but dwf_cg_schur are asynchronous on `stream`. */

/* out = Mooee in  /  out = Mooee^{-1} in  on a full (DWF_FULL) or half field of `parity`.  One read and
 * one write of the field (a thread walks the Ls slices of one 128-bit vector; Ls <= 32; larger Ls
 * re-reads).  in == out is allowed for Ls <= 32.  Errors: INVALID_ARG (NULL, misaligned, bad parity,
 * singular Mooee: M5 = 5 or 1 + mass (5-M5)^-Ls = 0), UNSUPPORTED (in == out with Ls > 32), CUDA. */
DWF_API int dwf_mooee(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass,
                      int dagger, void *stream);
DWF_API int dwf_mooee_inv(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass,
                          int dagger, void *stream);

/* out = M in on full fields (the unpreconditioned matrix): Mooee, then a x + b Dhop fused into the two
 * half-Dhop launches.  in != out.  Errors as dwf_dhop. */
DWF_API int dwf_ddwf(const dwf_geometry *g, const void *in_full, void *out_full, double M5, double mass, int dagger,
                     void *stream);

/* Schur complement of M on the sites of `parity` p (DWF_EVEN / DWF_ODD), q = 1 - p:
 *   S = Mooee - M_pq Mooee^{-1} M_qp = Mooee - 1/4 D_pq Mooee^{-1} D_qp        (in, out: half fields of parity p)
 * Four kernels: Dhop, Mooee^{-1}, Mooee, a x + b Dhop.  `work`: dwf_schur_work_bytes(g) bytes of device
 * memory owned by the caller (two half fields), 16-byte aligned.  in != out.  Errors as dwf_dhop_oe. */
DWF_API size_t dwf_schur_work_bytes(const dwf_geometry *g);
DWF_API int dwf_schur(const dwf_geometry *g, const void *in, void *out, int parity, double M5, double mass, int dagger,
                      void *work, void *stream);

/* out = a x + b y elementwise on fields of `parity` (any of x, y may be out). */
DWF_API int dwf_axpby(const dwf_geometry *g, double a, const void *x, double b, const void *y, void *out, int parity,
                      void *stream);

/* Solve S x = b on parity p by conjugate gradients on the normal equations S^dag S x = S^dag b, start
 * vector 0, in the geometry's precision (reductions in fp64).  Stops when |S^dag (b - S x)| <= tol |S^dag b|
 * (recursive residual) or after max_iter iterations; *iters_out = iterations done, *resid_out = the TRUE
 * relative residual |b - S x| / |b| recomputed at the end (either may be NULL).  `work`:
 * dwf_cg_work_bytes(g) bytes of device memory (six half fields).  Synchronises `stream` (two host
 * round trips per iteration for the step lengths).  Not reaching tol is not an error: check *resid_out. */
DWF_API size_t dwf_cg_work_bytes(const dwf_geometry *g);
DWF_API int dwf_cg_schur(const dwf_geometry *g, const void *b, void *x, int parity, double M5, double mass, double tol,
                         int max_iter, void *work, int *iters_out, double *resid_out, void *stream);

/* Bytes of a device field: full (DWF_FULL) or half (DWF_EVEN / DWF_ODD).  0 on bad arguments. */
DWF_API size_t dwf_field_bytes(const dwf_geometry *g, int parity);

/* canonical -> device layout.  Device sources are asynchronous on `stream`.  Host sources (pinned memory
 * for full PCIe speed) are moved in chunks of whole lattice lines through a ring of two 32 MB device
 * buffers: the H2D copy of chunk k+1 runs on an internal copy stream under the reorder kernel of chunk k;
 * the call synchronises `stream` before it returns unless the option "async_host" is set (then the host
 * array must stay untouched until dwf_host_wait). */
DWF_API int dwf_import_spinor(const dwf_geometry *g, const void *canonical, int src_is_device, int parity,
                      void *field_dev, void *stream);

/* device layout -> canonical.  Host destinations: the same ring in the other direction on a second copy
 * stream (an export's D2H copies overlap a following import's H2D copies: PCIe is full duplex); the call
 * waits for the last copy unless "async_host" is set (then the host array is complete after dwf_host_wait). */
DWF_API int dwf_export_spinor(const dwf_geometry *g, const void *field_dev, int parity, void *canonical,
                      int dst_is_device, void *stream);

/* Blocks until every host transfer (import / export with host arrays) issued on g has completed.  Only needed
 * with the option "async_host".  Errors: INVALID_ARG, CUDA. */
DWF_API int dwf_host_wait(const dwf_geometry *g);

/* Number of kernel launches this library has issued since it was loaded (all threads). */
DWF_API unsigned long long dwf_launch_count(void);

/* Name of the kernel a half-Dhop on this geometry runs with the current options, e.g.
 * "dhop_staged_kernel<16,4,2,2>" (Lh and the rows box of the tile), written NUL-terminated into
 * buf[0..n).  For reports; no effect on results.  Errors: INVALID_ARG. */
DWF_API int dwf_kernel_info(const dwf_geometry *g, char *buf, size_t n);

/* Tuning knobs for experiments; none of them changes a result of the staged kernel by a bit
 * (tests/test_gpu_staged.py).  UNSUPPORTED for an unknown key, INVALID_ARG for a bad value.
 *   "kernel"         0 auto, 1 direct (L1-cached) kernel, 2 TMA-staged kernel (error if it has no
 *                    variant for the geometry: Lh = L0/2 in {4, 8, 12, 16, 20, 24, 28, 32} (fp64: not 28), box extents
 *                    dividing L1..L3; other shapes run the direct kernel)
 *   "variant"        staged tile shape: 0 auto, n > 0 the n-th compiled (Lh, B1, B2, B3) instance
 *   "raster_staged"  launch order of the staged tiles, 10 * order + log2(macro blocks) (dhop_staged.cu); -1 auto
 *   "zigzag"         1: every other tile walks its s slices backwards (L2 reuse between tiles)
 *   "ssplit"         CTAs sharing one tile, each taking Ls / ssplit slices
 *   "layered"        1: one TMA box per x3 layer, so that L2 policies can differ per layer
 *   "l2pol"          decimal digits, one L2 eviction class per access type (dhop_staged.cu PC_*):
 *                    0 evict_normal, 1 evict_first, 2 evict_last
 *   "gauge12"        1: 12-real link storage (fp32 only): the NEXT dwf_load_gauge also keeps a copy
 *                    with rows 0, 1 of every link only, and dwf_dhop / dwf_dhop_oe / dwf_dhop_eo (the plain calls, on
 *                    geometries with a staged variant) read that copy and rebuild row 2 = conj(row0 x row1) once
 *                    per tile: 96 instead of 144 link bytes per 4D site and parity, model w (48 + 96/Ls) B per output
 *                    site.  The links must be SU(3) matrices; the result is the Dhop of the links with the rebuilt
 *                    third row (differs from the 18-real result by fp32 roundings of that row).  Until the reload
 *                    Dhop calls return NO_GAUGE.  UNSUPPORTED on fp64 geometries.
 *   "async_host"     1: dwf_import_spinor / dwf_export_spinor with host arrays return without synchronising
 *                    (pipelined steps; dwf_host_wait before touching the host arrays)
 *   "full_launch"    1 (default): dwf_dhop on an fp32 geometry with a staged variant is ONE launch whose tile table spans
 *                    both parities; 0: two half-field launches (same bits)
 *   "max_ctas"       > 0: cap on the number of CTAs of the staged kernels (0: one per SM, or two for small tiles).  Fewer
 *                    CTAs walk more tiles each: used by the tests of the tile switch on small lattices.
 *   "raster", "tile0".."tile3", "cpc"   direct kernel: CTA launch order, log2 tile extents, slices per CTA */
DWF_API int dwf_set_option(dwf_geometry *g, const char *key, long long value);

DWF_API const char *dwf_error_string(int code);
DWF_API const char *dwf_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DWF_H */

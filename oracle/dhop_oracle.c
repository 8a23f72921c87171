/*
 * oracle/dhop_oracle.c -- CPU ORACLE for the Domain Wall Fermion hopping term Dhop.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code, header, table or constant with the CUDA path
 * (paper_2203_06777_b200/csrc): the gamma matrices below are this file's own
 * copy, and the CUDA side never sees them.
 *
 * What it computes -- the plain definition of the operator the paper benchmarks
 * ("the Domain Wall Fermion operator", section 1; "node local
 * 'Wilson' matrix", L223 section 4; "main kernel DWF code", L254 Fig.6).  The
 * paper never prints the formula; BASELINE.json north_star states it and
 * SURVEY.md section 8(c) fixes every convention:
 *
 *   Dhop psi(x,s) = sum_{mu=0..3} [ (1 - gamma_mu) U_mu(x)        psi(x+mu,s)
 *                                 + (1 + gamma_mu) U_mu^dag(x-mu) psi(x-mu,s) ]
 *
 * evaluated exactly as written: full 4x4 spin matrices (NO half-spinor
 * projection trick), 3x3 complex colour mat-vec, fp64 arithmetic whatever the
 * storage precision of the inputs (fp32 inputs are promoted exactly), periodic
 * boundaries with an optional antiperiodic time direction (a hop that wraps
 * around mu=3 picks up a factor -1).  s is a pure spectator index.
 *
 * Pins (tests/test_oracle_pins.py): brute-force dense matrix assembled with
 * Kronecker products, free-field plane-wave closed form, gamma5-hermiticity,
 * gauge covariance, even/odd reassembly, s-equivariance, linearity,
 * translation covariance, norm bound.  Nothing here is "parity unpinned".
 *
 * Layouts (canonical / interchange, include/dwf.h):
 *   site    x = x0 + L0*(x1 + L1*(x2 + L2*x3)),   time = mu 3
 *   spinor  complex index ((site*Ls + s)*4 + spin)*3 + colour,  site = x (full
 *           field) or x>>1 (half field of one parity, sites in increasing x)
 *   gauge   complex index ((x*4 + mu)*3 + a)*3 + b  = U_mu(x)_{ab}, row a col b,
 *           (U psi)_a = sum_b U_ab psi_b
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* DeGrand-Rossi gamma matrices, mu = 0,1,2,3 = x,y,z,t. */
static const cplx GAMMA[4][4][4] = {
    { /* gamma_x */
        { 0, 0, 0, I },
        { 0, 0, I, 0 },
        { 0, -I, 0, 0 },
        { -I, 0, 0, 0 } },
    { /* gamma_y */
        { 0, 0, 0, -1 },
        { 0, 0, 1, 0 },
        { 0, 1, 0, 0 },
        { -1, 0, 0, 0 } },
    { /* gamma_z */
        { 0, 0, I, 0 },
        { 0, 0, 0, -I },
        { -I, 0, 0, 0 },
        { 0, I, 0, 0 } },
    { /* gamma_t */
        { 0, 0, 1, 0 },
        { 0, 0, 0, 1 },
        { 1, 0, 0, 0 },
        { 0, 1, 0, 0 } },
};

/* copy gamma_mu out as [4][4][2] reals, for the pins */
void orc_gamma(int mu, double *out)
{
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            out[(a * 4 + b) * 2]     = creal(GAMMA[mu][a][b]);
            out[(a * 4 + b) * 2 + 1] = cimag(GAMMA[mu][a][b]);
        }
}

/* Start-up self check: Hermitian, {g_mu,g_nu} = 2 delta, g5 = g0 g1 g2 g3 = diag(1,1,-1,-1).
 * Returns 0 when all three hold. */
int orc_check_gamma(void)
{
    for (int m = 0; m < 4; m++)
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++)
                if (cabs(GAMMA[m][a][b] - conj(GAMMA[m][b][a])) > 0) return 1;
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++)
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) {
                    cplx s = 0;
                    for (int c = 0; c < 4; c++)
                        s += GAMMA[m][a][c] * GAMMA[n][c][b] + GAMMA[n][a][c] * GAMMA[m][c][b];
                    cplx want = (m == n && a == b) ? 2.0 : 0.0;
                    if (cabs(s - want) > 0) return 2;
                }
    cplx g5[4][4], t[4][4];
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) g5[a][b] = GAMMA[0][a][b];
    for (int m = 1; m < 4; m++) {
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) {
                t[a][b] = 0;
                for (int c = 0; c < 4; c++) t[a][b] += g5[a][c] * GAMMA[m][c][b];
            }
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) g5[a][b] = t[a][b];
    }
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            cplx want = (a != b) ? 0.0 : (a < 2 ? 1.0 : -1.0);
            if (cabs(g5[a][b] - want) > 0) return 3;
        }
    return 0;
}

/* complex element k of an array of reals stored with `prec` bytes per real */
static inline cplx ldc(const void *p, int prec, size_t k)
{
    if (prec == 4) {
        const float *f = (const float *)p;
        return (double)f[2 * k] + I * (double)f[2 * k + 1];
    }
    const double *d = (const double *)p;
    return d[2 * k] + I * d[2 * k + 1];
}

typedef struct {
    int L[4];
    int Ls;
    int antiperiodic_t;
    const void *U;   int u_prec;
    const void *psi; int psi_prec;
    int psi_half;    /* 0: psi is a full field; 1: psi is a half field (index x>>1) */
    int dagger;      /* 0: Dhop; 1: Dhop^dagger */
} orc_ctx;

static inline size_t lex(const int L[4], const int x[4])
{
    return (size_t)x[0] + (size_t)L[0] * ((size_t)x[1] + (size_t)L[1] * ((size_t)x[2] + (size_t)L[2] * (size_t)x[3]));
}

static inline void coords(const int L[4], size_t site, int x[4])
{
    x[0] = (int)(site % (size_t)L[0]); site /= (size_t)L[0];
    x[1] = (int)(site % (size_t)L[1]); site /= (size_t)L[1];
    x[2] = (int)(site % (size_t)L[2]); site /= (size_t)L[2];
    x[3] = (int)site;
}

/* out[spin][colour] = (Dhop psi)(x, s), the definition written out term by term.
 * Dagger: the matrix adjoint of Dhop.  gamma_mu is Hermitian and the hop matrices W_mu, W_mu^dag
 * change places under the adjoint, so Dhop^dag has (1 + gamma_mu) on the forward hop and
 * (1 - gamma_mu) on the backward hop, with the same links. */
static void dhop_site(const orc_ctx *c, const int x[4], int s, cplx out[4][3])
{
    for (int al = 0; al < 4; al++)
        for (int a = 0; a < 3; a++) out[al][a] = 0;

    const size_t xs = lex(c->L, x);

    for (int mu = 0; mu < 4; mu++) {
        int xp[4] = { x[0], x[1], x[2], x[3] };
        int xm[4] = { x[0], x[1], x[2], x[3] };
        xp[mu] = (x[mu] + 1) % c->L[mu];
        xm[mu] = (x[mu] - 1 + c->L[mu]) % c->L[mu];
        double sp = 1.0, sm = 1.0;
        if (c->antiperiodic_t && mu == 3) {
            /* bc code 1: antiperiodic time, a wrapping hop gets -1.  bc code 2: OPEN time boundary (DESIGN.md
             * reading #26): a hop that would wrap contributes nothing -- the operator of one
             * time slab of a domain-decomposed lattice before the neighbours' faces are added. */
            const double w = (c->antiperiodic_t == 2) ? 0.0 : -1.0;
            if (x[3] == c->L[3] - 1) sp = w;   /* forward hop wraps  */
            if (x[3] == 0)           sm = w;   /* backward hop wraps */
        }
        const size_t xps = lex(c->L, xp), xms = lex(c->L, xm);
        const size_t ip = c->psi_half ? (xps >> 1) : xps;
        const size_t im = c->psi_half ? (xms >> 1) : xms;

        /* forward:  (1 - gamma_mu) U_mu(x) psi(x+mu, s) */
        cplx tf[4][3];
        for (int be = 0; be < 4; be++)
            for (int a = 0; a < 3; a++) {
                cplx acc = 0;
                for (int b = 0; b < 3; b++)
                    acc += ldc(c->U, c->u_prec, ((xs * 4 + (size_t)mu) * 3 + (size_t)a) * 3 + (size_t)b)
                         * ldc(c->psi, c->psi_prec, ((ip * (size_t)c->Ls + (size_t)s) * 4 + (size_t)be) * 3 + (size_t)b);
                tf[be][a] = acc;
            }
        /* backward: (1 + gamma_mu) U_mu^dag(x-mu) psi(x-mu, s),  U^dag_ab = conj(U_ba) */
        cplx tb[4][3];
        for (int be = 0; be < 4; be++)
            for (int a = 0; a < 3; a++) {
                cplx acc = 0;
                for (int b = 0; b < 3; b++)
                    acc += conj(ldc(c->U, c->u_prec, ((xms * 4 + (size_t)mu) * 3 + (size_t)b) * 3 + (size_t)a))
                         * ldc(c->psi, c->psi_prec, ((im * (size_t)c->Ls + (size_t)s) * 4 + (size_t)be) * 3 + (size_t)b);
                tb[be][a] = acc;
            }
        for (int al = 0; al < 4; al++)
            for (int be = 0; be < 4; be++) {
                cplx one = (al == be) ? 1.0 : 0.0;
                cplx pm = c->dagger ? one + GAMMA[mu][al][be] : one - GAMMA[mu][al][be];   /* forward hop  */
                cplx pp = c->dagger ? one - GAMMA[mu][al][be] : one + GAMMA[mu][al][be];   /* backward hop */
                for (int a = 0; a < 3; a++)
                    out[al][a] += sp * pm * tf[be][a] + sm * pp * tb[be][a];
            }
    }
}

static int bad_args(const int dims[4], int Ls, int u_prec, int psi_prec)
{
    if (Ls < 1) return 1;
    for (int m = 0; m < 4; m++) if (dims[m] < 1) return 1;
    if ((u_prec != 4 && u_prec != 8) || (psi_prec != 4 && psi_prec != 8)) return 1;
    return 0;
}

static void make_ctx(orc_ctx *c, const int dims[4], int Ls, int antiperiodic_t,
                     const void *U, int u_prec, const void *psi, int psi_prec, int psi_half)
{
    for (int m = 0; m < 4; m++) c->L[m] = dims[m];
    c->Ls = Ls; c->antiperiodic_t = antiperiodic_t;
    c->U = U; c->u_prec = u_prec; c->psi = psi; c->psi_prec = psi_prec; c->psi_half = psi_half;
    c->dagger = 0;
}

static void store_site(double *out, size_t osite, int Ls, int s, cplx r[4][3])
{
    for (int al = 0; al < 4; al++)
        for (int a = 0; a < 3; a++) {
            size_t k = ((osite * (size_t)Ls + (size_t)s) * 4 + (size_t)al) * 3 + (size_t)a;
            out[2 * k]     = creal(r[al][a]);
            out[2 * k + 1] = cimag(r[al][a]);
        }
}

/* Full Dhop: psi, out are full canonical fields (out always fp64). */
static int dhop_full(const int dims[4], int Ls, int antiperiodic_t, int dagger,
                     const void *U, int u_prec, const void *psi, int psi_prec, double *out)
{
    if (bad_args(dims, Ls, u_prec, psi_prec) || orc_check_gamma()) return 1;
    orc_ctx c; make_ctx(&c, dims, Ls, antiperiodic_t, U, u_prec, psi, psi_prec, 0);
    c.dagger = dagger;
    const int64_t V4 = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    #pragma omp parallel for schedule(static)
    for (int64_t site = 0; site < V4; site++) {
        int x[4]; coords(c.L, (size_t)site, x);
        for (int s = 0; s < Ls; s++) {
            cplx r[4][3];
            dhop_site(&c, x, s, r);
            store_site(out, (size_t)site, Ls, s, r);
        }
    }
    return 0;
}

/* Checkerboarded Dhop: output sites of parity `parity_out` only, psi is the half
 * field of the opposite parity, out the half field of parity_out (index x>>1).
 * parity_out = 1: DhopOE (even in -> odd out); parity_out = 0: DhopEO.
 * All extents must be even (x>>1 is a bijection within a parity only if L0 is even). */
static int dhop_cb(const int dims[4], int Ls, int antiperiodic_t, int parity_out, int dagger,
                   const void *U, int u_prec, const void *psi_half, int psi_prec, double *out_half)
{
    if (bad_args(dims, Ls, u_prec, psi_prec) || orc_check_gamma()) return 1;
    if (parity_out != 0 && parity_out != 1) return 1;
    for (int m = 0; m < 4; m++) if (dims[m] & 1) return 1;
    orc_ctx c; make_ctx(&c, dims, Ls, antiperiodic_t, U, u_prec, psi_half, psi_prec, 1);
    c.dagger = dagger;
    const int64_t V4 = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    #pragma omp parallel for schedule(static)
    for (int64_t site = 0; site < V4; site++) {
        int x[4]; coords(c.L, (size_t)site, x);
        if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity_out) continue;
        for (int s = 0; s < Ls; s++) {
            cplx r[4][3];
            dhop_site(&c, x, s, r);
            store_site(out_half, (size_t)site >> 1, Ls, s, r);
        }
    }
    return 0;
}

int orc_dhop(const int dims[4], int Ls, int antiperiodic_t,
             const void *U, int u_prec, const void *psi, int psi_prec, double *out)
{
    return dhop_full(dims, Ls, antiperiodic_t, 0, U, u_prec, psi, psi_prec, out);
}
int orc_dhop_dag(const int dims[4], int Ls, int antiperiodic_t,
                 const void *U, int u_prec, const void *psi, int psi_prec, double *out)
{
    return dhop_full(dims, Ls, antiperiodic_t, 1, U, u_prec, psi, psi_prec, out);
}
int orc_dhop_cb(const int dims[4], int Ls, int antiperiodic_t, int parity_out,
                const void *U, int u_prec, const void *psi_half, int psi_prec, double *out_half)
{
    return dhop_cb(dims, Ls, antiperiodic_t, parity_out, 0, U, u_prec, psi_half, psi_prec, out_half);
}
int orc_dhop_cb_dag(const int dims[4], int Ls, int antiperiodic_t, int parity_out,
                    const void *U, int u_prec, const void *psi_half, int psi_prec, double *out_half)
{
    return dhop_cb(dims, Ls, antiperiodic_t, parity_out, 1, U, u_prec, psi_half, psi_prec, out_half);
}

/* Dhop at a list of output sites (lexicographic indices), all s: out[n][Ls][4][3][2].
 * psi_half = 0: psi is a full field; 1: psi is the half field of the parity opposite
 * to every listed site (caller's responsibility).  Used to check sampled outputs at
 * sizes where a whole fp64 oracle field would not fit. */
int orc_dhop_sites(const int dims[4], int Ls, int antiperiodic_t,
                   const void *U, int u_prec, const void *psi, int psi_prec, int psi_half,
                   const int64_t *sites, int64_t n, double *out)
{
    if (bad_args(dims, Ls, u_prec, psi_prec) || orc_check_gamma()) return 1;
    orc_ctx c; make_ctx(&c, dims, Ls, antiperiodic_t, U, u_prec, psi, psi_prec, psi_half);
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; i++) {
        int x[4]; coords(c.L, (size_t)sites[i], x);
        for (int s = 0; s < Ls; s++) {
            cplx r[4][3];
            dhop_site(&c, x, s, r);
            store_site(out, (size_t)i, Ls, s, r);
        }
    }
    return 0;
}

/* sum |x_i|^2 over n reals, fp64 with Neumaier compensation (serial, fixed order) */
double orc_norm2(const void *x, int prec, int64_t n)
{
    double sum = 0.0, comp = 0.0;
    for (int64_t i = 0; i < n; i++) {
        double v = (prec == 4) ? (double)((const float *)x)[i] : ((const double *)x)[i];
        double t = v * v;
        double s = sum + t;
        comp += (fabs(sum) >= fabs(t)) ? (sum - s) + t : (t - s) + sum;
        sum = s;
    }
    return sum + comp;
}

/* sum conj(a_k) b_k over n complex numbers (2n reals each), compensated */
void orc_inner(const void *a, const void *b, int prec, int64_t ncomplex, double out[2])
{
    double sum[2] = { 0, 0 }, comp[2] = { 0, 0 };
    for (int64_t k = 0; k < ncomplex; k++) {
        cplx z = conj(ldc(a, prec, (size_t)k)) * ldc(b, prec, (size_t)k);
        double t[2] = { creal(z), cimag(z) };
        for (int j = 0; j < 2; j++) {
            double s = sum[j] + t[j];
            comp[j] += (fabs(sum[j]) >= fabs(t[j])) ? (sum[j] - s) + t[j] : (t[j] - s) + sum[j];
            sum[j] = s;
        }
    }
    out[0] = sum[0] + comp[0];
    out[1] = sum[1] + comp[1];
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

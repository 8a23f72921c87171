/*
 * oracle/dwf5d_oracle.c -- CPU ORACLE for the rest of the red-black Shamir domain-wall operator
 * ("5th-dimension term (chiral-projector hopping in s with the wall mass), its
 * inverse, ... the Schur complement").
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (same rules as dhop_oracle.c: only tests/, smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it; it shares nothing
 * with paper_2203_06777_b200/csrc).
 *
 * What it computes.  PAPER.md names the operator only ("all kernels involved in the DWF Dirac
 * operator", L223 section 4; L250 Fig.5, L254 Fig.6) and prints no formula; the definition used is
 * the standard Shamir domain-wall matrix, stated as reading #22 in DESIGN.md:
 *
 *   (M psi)(x,s) = (5 - M5) psi(x,s) - 1/2 (Dhop psi)(x,s) - P_- psi(x,s+1) - P_+ psi(x,s-1)
 *   P_+- = (1 +- gamma5)/2,   psi(x,Ls) := -m psi(x,0),   psi(x,-1) := -m psi(x,Ls-1)
 *
 * with Dhop the hopping term of dhop_oracle.c, M5 the domain-wall height, m the fermion mass.
 * "Mooee" is the part of M that is diagonal in the 4D site x (everything but Dhop); with the 4D
 * checkerboard of dhop_oracle.c, M = [Mee Meo; Moe Moo], Mee = Moo = Mooee, Meo = -1/2 DhopEO,
 * Moe = -1/2 DhopOE, and the Schur complement on parity p is
 *
 *   S_pp = Mooee - M_pq Mooee^{-1} M_qp              (q = 1 - p)
 *
 * How: nothing clever.  Mooee is assembled ONCE as a dense real (4 Ls) x (4 Ls) matrix straight
 * from the formula above (full 4x4 projectors from this oracle's own gamma matrices, index
 * s*4 + spin), and the four operations a solver needs are dense linear algebra on it: apply A,
 * apply A^T (the adjoint: A is real), apply inv(A), apply inv(A)^T, the inverse by Gauss-Jordan
 * elimination with partial pivoting.  The CUDA path uses chirality-split recurrences in s instead.
 * M and S are compositions of these with the whole-field Dhop entry points of dhop_oracle.c.
 *
 * Pins (tests/test_oracle_pins_dwf.py): dense matrix over (x, s, spin, colour) assembled with
 * Kronecker products in numpy, numpy.linalg inverse / Schur complement of that matrix,
 * Mooee Mooee^{-1} = 1, gamma5 R5-hermiticity, Ls = 1 and m = -1 / +1 (periodic / antiperiodic s)
 * closed forms.  Nothing here is "parity unpinned".
 *
 * Layouts: canonical spinor [site][s][spin][colour][reim] (include/dwf.h); outputs always fp64.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* entry points of dhop_oracle.c used here */
void orc_gamma(int mu, double *out);
int orc_dhop(const int dims[4], int Ls, int antiperiodic_t, const void *U, int u_prec, const void *psi, int psi_prec, double *out);
int orc_dhop_dag(const int dims[4], int Ls, int antiperiodic_t, const void *U, int u_prec, const void *psi, int psi_prec, double *out);
int orc_dhop_cb(const int dims[4], int Ls, int antiperiodic_t, int parity_out, const void *U, int u_prec, const void *psi_half, int psi_prec, double *out_half);
int orc_dhop_cb_dag(const int dims[4], int Ls, int antiperiodic_t, int parity_out, const void *U, int u_prec, const void *psi_half, int psi_prec, double *out_half);

enum { ORC_M5 = 0, ORC_M5_DAG = 1, ORC_M5_INV = 2, ORC_M5_INV_DAG = 3 };

/* gamma5 = gamma0 gamma1 gamma2 gamma3 from the oracle's own table; must come out real */
static int gamma5_real(double g5[4][4])
{
    double a[4][4][2], b[4][4][2], t[4][4][2];
    orc_gamma(0, &a[0][0][0]);
    for (int mu = 1; mu < 4; mu++) {
        orc_gamma(mu, &b[0][0][0]);
        for (int i = 0; i < 4; i++)
            for (int j = 0; j < 4; j++) {
                double re = 0, im = 0;
                for (int k = 0; k < 4; k++) {
                    re += a[i][k][0] * b[k][j][0] - a[i][k][1] * b[k][j][1];
                    im += a[i][k][0] * b[k][j][1] + a[i][k][1] * b[k][j][0];
                }
                t[i][j][0] = re; t[i][j][1] = im;
            }
        memcpy(a, t, sizeof(a));
    }
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            if (a[i][j][1] != 0.0) return 1;
            g5[i][j] = a[i][j][0];
        }
    return 0;
}

/* A[(s,al),(s',be)] of Mooee, n = 4 Ls, row-major, exactly the formula in the header */
static int build_mooee(int Ls, double M5, double mass, double *A)
{
    const int n = 4 * Ls;
    double g5[4][4], Pp[4][4], Pm[4][4];
    if (gamma5_real(g5)) return 1;
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            const double one = (i == j) ? 1.0 : 0.0;
            Pp[i][j] = 0.5 * (one + g5[i][j]);
            Pm[i][j] = 0.5 * (one - g5[i][j]);
        }
    memset(A, 0, sizeof(double) * (size_t)n * (size_t)n);
    for (int s = 0; s < Ls; s++)
        for (int al = 0; al < 4; al++) {
            const int r = s * 4 + al;
            A[(size_t)r * n + r] += 5.0 - M5;
            /* - P_- psi(s+1), psi(Ls) = -m psi(0) */
            int sp = s + 1; double cp = -1.0;
            if (sp == Ls) { sp = 0; cp = mass; }
            /* - P_+ psi(s-1), psi(-1) = -m psi(Ls-1) */
            int sm = s - 1; double cm = -1.0;
            if (sm < 0) { sm = Ls - 1; cm = mass; }
            for (int be = 0; be < 4; be++) {
                A[(size_t)r * n + (sp * 4 + be)] += cp * Pm[al][be];
                A[(size_t)r * n + (sm * 4 + be)] += cm * Pp[al][be];
            }
        }
    return 0;
}

/* in-place inverse by Gauss-Jordan elimination with partial pivoting; returns 1 if singular */
static int invert(int n, double *A)
{
    double *W = (double *)malloc(sizeof(double) * (size_t)n * 2 * (size_t)n);
    if (!W) return 1;
    for (int i = 0; i < n; i++)
        for (int j = 0; j < 2 * n; j++)
            W[(size_t)i * 2 * n + j] = (j < n) ? A[(size_t)i * n + j] : ((j - n == i) ? 1.0 : 0.0);
    for (int c = 0; c < n; c++) {
        int piv = c;
        for (int i = c + 1; i < n; i++)
            if (fabs(W[(size_t)i * 2 * n + c]) > fabs(W[(size_t)piv * 2 * n + c])) piv = i;
        if (W[(size_t)piv * 2 * n + c] == 0.0) { free(W); return 1; }
        if (piv != c)
            for (int j = 0; j < 2 * n; j++) {
                double t = W[(size_t)c * 2 * n + j];
                W[(size_t)c * 2 * n + j] = W[(size_t)piv * 2 * n + j];
                W[(size_t)piv * 2 * n + j] = t;
            }
        const double d = W[(size_t)c * 2 * n + c];
        for (int j = 0; j < 2 * n; j++) W[(size_t)c * 2 * n + j] /= d;
        for (int i = 0; i < n; i++) {
            if (i == c) continue;
            const double f = W[(size_t)i * 2 * n + c];
            if (f == 0.0) continue;
            for (int j = 0; j < 2 * n; j++) W[(size_t)i * 2 * n + j] -= f * W[(size_t)c * 2 * n + j];
        }
    }
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) A[(size_t)i * n + j] = W[(size_t)i * 2 * n + n + j];
    free(W);
    return 0;
}

static inline double ldr(const void *p, int prec, size_t k)
{
    return prec == 4 ? (double)((const float *)p)[k] : ((const double *)p)[k];
}

/* copy the dense (4 Ls)^2 matrix of operation `op` out, for the pins */
int orc_mooee_matrix(int Ls, double M5, double mass, int op, double *out)
{
    if (Ls < 1 || op < 0 || op > 3) return 1;
    const int n = 4 * Ls;
    double *A = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    if (!A || build_mooee(Ls, M5, mass, A)) { free(A); return 1; }
    if (op >= 2 && invert(n, A)) { free(A); return 1; }
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++)
            out[(size_t)i * n + j] = (op & 1) ? A[(size_t)j * n + i] : A[(size_t)i * n + j];
    free(A);
    return 0;
}

/* out(x, s, al, c) = sum_{s', be} Op[(s,al),(s',be)] in(x, s', be, c) for every site x of the
 * field (nsites of them: a full field or a half field -- Mooee does not couple sites). */
int orc_mooee(int64_t nsites, int Ls, double M5, double mass, int op, const void *in, int prec, double *out)
{
    if (nsites < 0 || Ls < 1 || op < 0 || op > 3 || (prec != 4 && prec != 8)) return 1;
    const int n = 4 * Ls;
    double *A = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    if (!A || orc_mooee_matrix(Ls, M5, mass, op, A)) { free(A); return 1; }
    #pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < nsites; x++) {
        const size_t base = (size_t)x * (size_t)n * 6;          /* reals: [s*4+al][colour][reim] */
        for (int r = 0; r < n; r++) {
            double acc[6] = { 0, 0, 0, 0, 0, 0 };
            for (int q = 0; q < n; q++) {
                const double a = A[(size_t)r * n + q];
                if (a == 0.0) continue;
                for (int k = 0; k < 6; k++) acc[k] += a * ldr(in, prec, base + (size_t)q * 6 + k);
            }
            for (int k = 0; k < 6; k++) out[base + (size_t)r * 6 + k] = acc[k];
        }
    }
    free(A);
    return 0;
}

/* Full Shamir DWF matrix on a full field: out = Mooee psi - 1/2 Dhop psi (dagger: the adjoint) */
int orc_ddwf(const int dims[4], int Ls, int antiperiodic_t, double M5, double mass, int dagger,
             const void *U, int u_prec, const void *psi, int psi_prec, double *out)
{
    const int64_t V4 = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    const size_t n = (size_t)V4 * (size_t)Ls * 24;
    double *t = (double *)malloc(sizeof(double) * n);
    if (!t) return 1;
    int rc = dagger ? orc_dhop_dag(dims, Ls, antiperiodic_t, U, u_prec, psi, psi_prec, t)
                    : orc_dhop(dims, Ls, antiperiodic_t, U, u_prec, psi, psi_prec, t);
    if (!rc) rc = orc_mooee(V4, Ls, M5, mass, dagger ? ORC_M5_DAG : ORC_M5, psi, psi_prec, out);
    if (!rc)
        for (size_t i = 0; i < n; i++) out[i] -= 0.5 * t[i];
    free(t);
    return rc;
}

/* Schur complement on parity p (psi, out: half fields of parity p):
 *   S   = Mooee     - M_pq     Mooee^{-1}  M_qp,      M_qp = -1/2 D_qp (input parity p -> output parity q)
 *   S^+ = Mooee^+   - M_qp^+   Mooee^{-+}  M_pq^+,    M_pq^+ = -1/2 (D^+)_qp
 * evaluated right to left exactly as written. */
int orc_schur(const int dims[4], int Ls, int antiperiodic_t, double M5, double mass, int dagger, int parity,
              const void *U, int u_prec, const void *psi_half, int psi_prec, double *out_half)
{
    if (parity != 0 && parity != 1) return 1;
    const int64_t Vh = (int64_t)dims[0] * dims[1] * dims[2] * dims[3] / 2;
    const size_t n = (size_t)Vh * (size_t)Ls * 24;
    const int q = 1 - parity;
    double *t = (double *)malloc(sizeof(double) * n), *u = (double *)malloc(sizeof(double) * n);
    int rc = (!t || !u);
    /* t_q = -1/2 D_qp psi_p */
    if (!rc) rc = dagger ? orc_dhop_cb_dag(dims, Ls, antiperiodic_t, q, U, u_prec, psi_half, psi_prec, t)
                         : orc_dhop_cb(dims, Ls, antiperiodic_t, q, U, u_prec, psi_half, psi_prec, t);
    if (!rc) for (size_t i = 0; i < n; i++) t[i] *= -0.5;
    /* u_q = Mooee^{-1} t_q */
    if (!rc) rc = orc_mooee(Vh, Ls, M5, mass, dagger ? ORC_M5_INV_DAG : ORC_M5_INV, t, 8, u);
    /* t_p = -1/2 D_pq u_q */
    if (!rc) rc = dagger ? orc_dhop_cb_dag(dims, Ls, antiperiodic_t, parity, U, u_prec, u, 8, t)
                         : orc_dhop_cb(dims, Ls, antiperiodic_t, parity, U, u_prec, u, 8, t);
    if (!rc) for (size_t i = 0; i < n; i++) t[i] *= -0.5;
    /* out = Mooee psi_p - t_p */
    if (!rc) rc = orc_mooee(Vh, Ls, M5, mass, dagger ? ORC_M5_DAG : ORC_M5, psi_half, psi_prec, out_half);
    if (!rc) for (size_t i = 0; i < n; i++) out_half[i] -= t[i];
    free(t); free(u);
    return rc;
}

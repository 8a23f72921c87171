/*
 * dwf_inputs/gen.c -- seeded synthetic input generators (gauge fields, spinors).
 *
 * This module serves BOTH the CPU oracle tests and the CUDA path.  It holds none
 * of the Dhop arithmetic: it only fills arrays with seeded random data in the
 * canonical (interchange) layouts of include/dwf.h.  Recipes follow SURVEY.md
 * section 8(c) readings #12-#15 (BASELINE.json "configs"):
 *
 *   - counter-based RNG: value(seed, stream, element) is a pure function, so the
 *     output does not depend on thread count or generation order;
 *   - Gaussian spinor: re and im parts iid N(0,1), Box-Muller;
 *   - random SU(3): 3x3 complex Gaussian matrix, modified Gram-Schmidt on rows
 *     0,1,2, then row 2 multiplied by conj(det) so that det = 1;
 *   - near-unit SU(3): U = exp(i*eps*H), H random traceless Hermitian, Taylor
 *     series in fp64, then the same Gram-Schmidt + det fix.
 *
 * Everything is computed in fp64 and rounded once on output when prec == 4.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <complex.h>

typedef double complex cplx;

static inline uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* uniform in (0,1), never 0 or 1 */
static inline double uniform01(uint64_t key, uint64_t counter)
{
    uint64_t r = mix64(key + counter * 0xD1342543DE82EF95ULL);
    return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

static inline uint64_t stream_key(uint64_t seed, uint64_t stream)
{
    return mix64(mix64(seed) ^ (stream * 0xA24BAED4963EE407ULL + 0x632BE59BD9B4E019ULL));
}

/* element e of the N(0,1) sequence of (seed, stream) */
static inline double gaussian(uint64_t key, uint64_t e)
{
    uint64_t pair = e >> 1;
    double u1 = uniform01(key, 2 * pair);
    double u2 = uniform01(key, 2 * pair + 1);
    double r = sqrt(-2.0 * log(u1));
    double a = 6.283185307179586476925286766559 * u2;
    return (e & 1) ? r * sin(a) : r * cos(a);
}

static inline void store_real(void *out, int prec, size_t idx, double v)
{
    if (prec == 4) ((float *)out)[idx] = (float)v;
    else           ((double *)out)[idx] = v;
}

/* n reals, iid N(0,1); element index offset `first` lets callers fill slabs */
int dwfin_gaussian(uint64_t seed, uint64_t stream, uint64_t first, uint64_t n,
                   int prec, void *out)
{
    if ((prec != 4 && prec != 8) || !out) return 1;
    uint64_t key = stream_key(seed, stream);
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; i++)
        store_real(out, prec, (size_t)i, gaussian(key, first + (uint64_t)i));
    return 0;
}

/* rows 0,1,2 orthonormalised in order (modified Gram-Schmidt), then det -> 1 */
static void project_su3(cplx m[3][3])
{
    for (int r = 0; r < 3; r++) {
        for (int q = 0; q < r; q++) {
            cplx dot = 0;
            for (int c = 0; c < 3; c++) dot += conj(m[q][c]) * m[r][c];
            for (int c = 0; c < 3; c++) m[r][c] -= dot * m[q][c];
        }
        double nrm = 0;
        for (int c = 0; c < 3; c++) nrm += creal(m[r][c] * conj(m[r][c]));
        nrm = 1.0 / sqrt(nrm);
        for (int c = 0; c < 3; c++) m[r][c] *= nrm;
    }
    cplx det = m[0][0] * (m[1][1] * m[2][2] - m[1][2] * m[2][1])
             - m[0][1] * (m[1][0] * m[2][2] - m[1][2] * m[2][0])
             + m[0][2] * (m[1][0] * m[2][1] - m[1][1] * m[2][0]);
    for (int c = 0; c < 3; c++) m[2][c] *= conj(det);
}

static void store_link(void *out, int prec, uint64_t link, cplx m[3][3])
{
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) {
            size_t idx = ((size_t)link * 9 + (size_t)(a * 3 + b)) * 2;
            store_real(out, prec, idx,     creal(m[a][b]));
            store_real(out, prec, idx + 1, cimag(m[a][b]));
        }
}

/* nlinks random SU(3) matrices, link index offset `first` */
int dwfin_su3_random(uint64_t seed, uint64_t stream, uint64_t first, uint64_t nlinks,
                     int prec, void *out)
{
    if ((prec != 4 && prec != 8) || !out) return 1;
    uint64_t key = stream_key(seed, stream);
    #pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)nlinks; l++) {
        uint64_t g = (first + (uint64_t)l) * 18;
        cplx m[3][3];
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                int k = (a * 3 + b) * 2;
                m[a][b] = gaussian(key, g + k) + I * gaussian(key, g + k + 1);
            }
        project_su3(m);
        store_link(out, prec, (uint64_t)l, m);
    }
    return 0;
}

/* nlinks matrices U = exp(i*eps*H), H random traceless Hermitian, projected to SU(3) */
int dwfin_su3_near_unit(uint64_t seed, uint64_t stream, uint64_t first, uint64_t nlinks,
                        double eps, int prec, void *out)
{
    if ((prec != 4 && prec != 8) || !out) return 1;
    uint64_t key = stream_key(seed, stream);
    #pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)nlinks; l++) {
        uint64_t g = (first + (uint64_t)l) * 18;
        cplx G[3][3], A[3][3], T[3][3], U[3][3], N[3][3];
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                int k = (a * 3 + b) * 2;
                G[a][b] = gaussian(key, g + k) + I * gaussian(key, g + k + 1);
            }
        /* H = (G + G^dag)/2 - tr/3 ;  A = i*eps*H */
        cplx tr = 0;
        for (int a = 0; a < 3; a++) tr += 0.5 * (G[a][a] + conj(G[a][a]));
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                cplx h = 0.5 * (G[a][b] + conj(G[b][a]));
                if (a == b) h -= tr / 3.0;
                A[a][b] = I * eps * h;
            }
        /* U = sum_k A^k / k!, 30 terms */
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                U[a][b] = (a == b) ? 1.0 : 0.0;
                T[a][b] = U[a][b];
            }
        for (int k = 1; k <= 30; k++) {
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) {
                    cplx s = 0;
                    for (int c = 0; c < 3; c++) s += T[a][c] * A[c][b];
                    N[a][b] = s / (double)k;
                }
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) {
                    T[a][b] = N[a][b];
                    U[a][b] += T[a][b];
                }
        }
        project_su3(U);
        store_link(out, prec, (uint64_t)l, U);
    }
    return 0;
}

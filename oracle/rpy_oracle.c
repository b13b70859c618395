/*
 * rpy_oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, obviously-correct float64 CPU statement of what the hot path of
 * arXiv:1602.02170 computes: the blob-blob mobility product  u = M lambda
 * (Eq. (6)) by direct O(N_b^2) summation,
 * with M the Rotne-Prager-Yamakawa tensor, Eq. (9), and,
 * for blobs above a single no-slip wall at z = 0, the translation-translation
 * Rotne-Prager-Blake wall correction added to it.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this file.  It shares no code, header, table or
 * constant with the CUDA path under paper_1602_02170_b200/csrc/.
 *
 * Reading of the paper where it is silent:
 *  - the wall block is Eq. (7) applied to the image part of
 *    Blake's half-space Green's function [72]; the paper cites [13] (B1),(C2)
 *    for the result instead of printing it.  The closed form written out in
 *    wall_block() below is pinned by tests/test_oracle_wall.py against an
 *    independent finite-difference evaluation of Eq. (7) on Blake's tensor.
 *  - r <= 2a takes the overlap branch (Eq. (9)); r = 0 gives the identity
 *    block, dyad defined as 0.
 *  - the wall block is added for every pair, including i = j and overlapping
 *    pairs (overlap corrections are independent of the wall).
 *  - one radius a and one viscosity eta for all blobs; prefactor 1/(6 pi eta a)
 *    on the RPY block, 1/(8 pi eta) = (1/(6 pi eta a)) (3a/4) on W.
 *
 * Arithmetic: float64 with sqrt and division, no reordering; the row sums are
 * accumulated in long double (x87 80-bit here) so that the oracle's own
 * summation error stays ~1e-19 of sum|terms|.  Rows are independent; OpenMP is
 * used over rows only and the inner loop is the plain definition.
 *
 * Pins: every exported function is pinned (tests/test_oracle_*.py, -m "not gpu").
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define RPY_ORACLE_FREE 0
#define RPY_ORACLE_WALL 1

static const double PI = 3.14159265358979323846264338327950288;

/* Eq. (9): dimensionless block 6 pi eta a * M_ij for
 * r_ij = r_i - r_j.  B is row-major 3x3. */
static void rpy_block(const double ri[3], const double rj[3], double a, double B[9])
{
    double d[3] = { ri[0] - rj[0], ri[1] - rj[1], ri[2] - rj[2] };
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double cI, cD;           /* coefficient of I and of rhat (x) rhat */
    double rh[3] = { 0.0, 0.0, 0.0 };
    if (r > 0.0) { rh[0] = d[0] / r; rh[1] = d[1] / r; rh[2] = d[2] / r; }
    if (r > 2.0 * a) {
        double x = a / r;
        cI = 3.0 * x / 4.0 + x * x * x / 2.0;        /* C1 */
        cD = 3.0 * x / 4.0 - 3.0 * x * x * x / 2.0;  /* C2 */
    } else {
        cI = 1.0 - 9.0 * r / (32.0 * a);             /* C3 */
        cD = 3.0 * r / (32.0 * a);                   /* C4 */
    }
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q)
            B[3 * p + q] = (p == q ? cI : 0.0) + cD * rh[p] * rh[q];
}

/* Wall block (3a/4) W(r_i, r_j), dimensionless (units of 1/(6 pi eta a)).
 * W = 8 pi (1 + a^2/6 lap_i)(1 + a^2/6 lap_j)[G_Blake - Oseen], Eq. (7) with
 * Blake's image system.  Row = velocity component at
 * blob i, column = force component at blob j.  Notation of SURVEY.md 8(c):
 * R = (x_i-x_j, y_i-y_j, z_i+z_j), e = R/|R|, Greek indices in {x,y}. */
static void wall_block(const double ri[3], const double rj[3], double a, double B[9])
{
    double zi = ri[2], zj = rj[2];
    double Rv[3] = { ri[0] - rj[0], ri[1] - rj[1], zi + zj };
    double R = sqrt(Rv[0] * Rv[0] + Rv[1] * Rv[1] + Rv[2] * Rv[2]);
    double e[3] = { Rv[0] / R, Rv[1] / R, Rv[2] / R };
    double ez2 = e[2] * e[2], ez4 = ez2 * ez2;
    double R3 = R * R * R, R5 = R3 * R * R;
    double a2 = a * a, a4 = a2 * a2;
    double W[9];

    for (int al = 0; al < 2; ++al)
        for (int be = 0; be < 2; ++be) {
            double dl = (al == be) ? 1.0 : 0.0;
            double ee = e[al] * e[be];
            W[3 * al + be] =
                -(dl + ee) / R
                - 2.0 * zi * zj * (dl - 3.0 * ee) / R3
                + a2 * (-(2.0 / 3.0) * (1.0 - 3.0 * ez2) * dl + 2.0 * (1.0 - 5.0 * ez2) * ee) / R3
                + a4 * ((2.0 / 3.0) * (1.0 - 5.0 * ez2) * dl - (10.0 / 3.0) * (1.0 - 7.0 * ez2) * ee) / R5;
        }
    W[8] = -(1.0 + ez2) / R
           + 2.0 * zi * zj * (1.0 - 3.0 * ez2) / R3
           - (2.0 / 3.0) * a2 * (1.0 + 6.0 * ez2 - 15.0 * ez4) / R3
           - (2.0 / 3.0) * a4 * (3.0 - 30.0 * ez2 + 35.0 * ez4) / R5;
    double t1 = (zj - zi) / (R * R);
    double t2 = 6.0 * e[2] * zi * zj / R3
              + 2.0 * a2 * e[2] * (1.0 - 5.0 * ez2) / R3
              - (10.0 / 3.0) * a4 * e[2] * (3.0 - 7.0 * ez2) / R5;
    for (int al = 0; al < 2; ++al) {
        W[3 * al + 2] = e[al] * (t1 - t2);   /* velocity alpha at i, force z at j */
        W[6 + al]     = e[al] * (t1 + t2);   /* velocity z at i, force alpha at j */
    }
    for (int q = 0; q < 9; ++q) B[q] = (3.0 * a / 4.0) * W[q];
}

/* M_ij as a row-major 3x3 block, dimensional: (1/(6 pi eta a)) [RPY (+ wall)].
 * variant: RPY_ORACLE_FREE or RPY_ORACLE_WALL. */
void rpy_oracle_pair(int variant, const double ri[3], const double rj[3],
                     double a, double eta, double M[9])
{
    double B[9], Wb[9];
    double pref = 1.0 / (6.0 * PI * eta * a);
    rpy_block(ri, rj, a, B);
    if (variant == RPY_ORACLE_WALL) {
        wall_block(ri, rj, a, Wb);
        for (int q = 0; q < 9; ++q) B[q] += Wb[q];
    }
    for (int q = 0; q < 9; ++q) M[q] = pref * B[q];
}

/* The wall block alone, dimensionless: (3a/4) W(r_i, r_j) = 6 pi eta a (M_wall - M_free). */
void rpy_oracle_wall_block(const double ri[3], const double rj[3], double a, double B[9])
{
    wall_block(ri, rj, a, B);
}

/* Dense mobility matrix, row-major (3n) x (3n): block (i,j) at rows 3i..3i+2,
 * columns 3j..3j+2 (block layout of PAPER.md:120).  pos is [n][3]. */
void rpy_oracle_dense(int variant, int64_t n, const double *pos, double a, double eta, double *M)
{
    int64_t ld = 3 * n;
    for (int64_t i = 0; i < n; ++i)
        for (int64_t j = 0; j < n; ++j) {
            double B[9];
            rpy_oracle_pair(variant, pos + 3 * i, pos + 3 * j, a, eta, B);
            for (int p = 0; p < 3; ++p)
                for (int q = 0; q < 3; ++q)
                    M[(3 * i + p) * ld + (3 * j + q)] = B[3 * p + q];
        }
}

/* u_i = sum_{j=0..n-1} M_ij lambda_j  (all j including j = i), Eq. (6), for the
 * requested target rows.
 *   pos   [n][3], force [k][n][3], rows [nrows] (NULL => rows 0..nrows-1),
 *   vel   [k][nrows][3] (overwritten).
 * The sum over j runs in index order; each M_ij is formed as the full 3x3 block
 * and multiplied, no use of structure. */
void rpy_oracle_matvec(int variant, int64_t n, int k, const double *pos, const double *force,
                       double a, double eta, int64_t nrows, const int64_t *rows, double *vel)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 4)
#endif
    for (int64_t ir = 0; ir < nrows; ++ir) {
        int64_t i = rows ? rows[ir] : ir;
        long double acc[3 * k];                 /* one running sum per (rhs, component) */
        for (int q = 0; q < 3 * k; ++q) acc[q] = 0.0L;
        for (int64_t j = 0; j < n; ++j) {
            double B[9];
            rpy_oracle_pair(variant, pos + 3 * i, pos + 3 * j, a, eta, B);
            for (int s = 0; s < k; ++s) {
                const double *lam = force + ((size_t)s * n + j) * 3;
                for (int p = 0; p < 3; ++p)
                    acc[3 * s + p] += (long double)B[3 * p + 0] * lam[0]
                                    + (long double)B[3 * p + 1] * lam[1]
                                    + (long double)B[3 * p + 2] * lam[2];
            }
        }
        for (int s = 0; s < k; ++s)
            for (int p = 0; p < 3; ++p)
                vel[((size_t)s * nrows + ir) * 3 + p] = (double)acc[3 * s + p];
    }
}

/* Flow field, Appendix B: v(r_t) = sum_j M'(r_t, r_j) lambda'_j at targets that
 * are not the sources; M' is the same pair tensor with the tracer radius as `a` (both blobs of the
 * pair have that radius).  tgt [nt][3], src [ns][3], force [k][ns][3], vel [k][nt][3]. */
void rpy_oracle_flow(int variant, int64_t nt, const double *tgt, int64_t ns, const double *src, int k,
                     const double *force, double a, double eta, double *vel)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 4)
#endif
    for (int64_t t = 0; t < nt; ++t) {
        long double acc[3 * k];
        for (int q = 0; q < 3 * k; ++q) acc[q] = 0.0L;
        for (int64_t j = 0; j < ns; ++j) {
            double B[9];
            rpy_oracle_pair(variant, tgt + 3 * t, src + 3 * j, a, eta, B);
            for (int s = 0; s < k; ++s) {
                const double *lam = force + ((size_t)s * ns + j) * 3;
                for (int p = 0; p < 3; ++p)
                    acc[3 * s + p] += (long double)B[3 * p + 0] * lam[0]
                                    + (long double)B[3 * p + 1] * lam[1]
                                    + (long double)B[3 * p + 2] * lam[2];
            }
        }
        for (int s = 0; s < k; ++s)
            for (int p = 0; p < 3; ++p)
                vel[((size_t)s * nt + t) * 3 + p] = (double)acc[3 * s + p];
    }
}

/* Threads the row loop actually uses (reported beside the timed baseline). */
int rpy_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

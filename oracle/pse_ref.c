/* pse_ref.c — inner loops of the fp64 CPU PSE reference (oracle/pse_reference.py).  TEST INFRASTRUCTURE ONLY:
 * nothing under paper_1709_06946_b200/ includes, links or calls this file, and it includes nothing from there.
 *
 * Plain C + OpenMP, no blocking or fusion beyond what the paper states:
 *   ref_spread       Q   : g_c(x_n) = sum_beta K(x_n - x_beta) q_{beta,c}       (Gaussian K PAPER.md:263)
 *   ref_interp       Q^T : out_{alpha,c} = sum_n K(x_n - x_alpha) g_c(x_n)      (the h^3 is applied by the caller)
 *   ref_pairs        M_r : cut-off pair sum over linked cells of edge >= r_cut, tensor forms of
 *                          Eqs. (25)-(27) in the notation of SURVEY.md 8(c) O4, self term O5
 * The Gaussian on the grid is exp(-(2 pi / P) t^2), t = distance in grid spacings (eta_g = (h P xi / m)^2, m = sqrt(pi P),
 * PAPER.md:306, 334); its normalisation (2 xi^2/(pi eta_g))^{3/2} is applied by the caller.
 * Support placement (reading R5): odd P centred on the nearest grid point, even P base = floor(x/h) - P/2 + 1.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int ref_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static long support_base(double g, int P) { return (P & 1) ? lround(g) - (P - 1) / 2 : (long)floor(g) - P / 2 + 1; }
static int pmod(long i, int M) { long r = i % M; return (int)(r < 0 ? r + M : r); }

static void weights(const double *x, double inv_h, int P, int M, long base[3], double w[3][64], int idx[3][64]) {
    const double c = 2.0 * M_PI / P;
    for (int d = 0; d < 3; ++d) {
        const double g = x[d] * inv_h;
        base[d] = support_base(g, P);
        for (int i = 0; i < P; ++i) {
            const double t = (double)(base[d] + i) - g;
            w[d][i] = exp(-c * t * t);
            idx[d][i] = pmod(base[d] + i, M);
        }
    }
}

/* x [N][3], q [N][C], grid [C][M][M][M] (zeroed here).  Threads own disjoint ranges of grid x-planes and each walks all
 * particles, so no two threads ever write the same grid value and the summation order is the particle order. */
void ref_spread(int N, const double *x, const double *q, int C, int M, int P, double L, double *grid) {
    const double inv_h = M / L;
    const size_t M3 = (size_t)M * M * M;
    memset(grid, 0, sizeof(double) * M3 * C);
#pragma omp parallel
    {
#ifdef _OPENMP
        const int nt = omp_get_num_threads(), me = omp_get_thread_num();
#else
        const int nt = 1, me = 0;
#endif
        const int lo = (int)((long)M * me / nt), hi = (int)((long)M * (me + 1) / nt);
        long base[3]; double w[3][64]; int idx[3][64];
        for (int b = 0; b < N; ++b) {
            weights(x + 3 * (size_t)b, inv_h, P, M, base, w, idx);
            for (int i = 0; i < P; ++i) {
                const int gx = idx[0][i];
                if (gx < lo || gx >= hi) continue;
                for (int j = 0; j < P; ++j) {
                    const double wxy = w[0][i] * w[1][j];
                    const size_t row = ((size_t)gx * M + idx[1][j]) * M;
                    for (int k = 0; k < P; ++k) {
                        const double ww = wxy * w[2][k];
                        for (int c = 0; c < C; ++c) grid[c * M3 + row + idx[2][k]] += ww * q[(size_t)b * C + c];
                    }
                }
            }
        }
    }
}

/* rows [nrows] particle indices; out [nrows][C] */
void ref_interp(int nrows, const long *rows, const double *x, int C, int M, int P, double L, const double *grid, double *out) {
    const double inv_h = M / L;
    const size_t M3 = (size_t)M * M * M;
#pragma omp parallel for schedule(static)
    for (int r = 0; r < nrows; ++r) {
        long base[3]; double w[3][64]; int idx[3][64];
        weights(x + 3 * (size_t)rows[r], inv_h, P, M, base, w, idx);
        double acc[16];
        for (int c = 0; c < C; ++c) acc[c] = 0.0;
        for (int i = 0; i < P; ++i)
            for (int j = 0; j < P; ++j) {
                const double wxy = w[0][i] * w[1][j];
                const size_t row = ((size_t)idx[0][i] * M + idx[1][j]) * M;
                for (int k = 0; k < P; ++k) {
                    const double ww = wxy * w[2][k];
                    for (int c = 0; c < C; ++c) acc[c] += ww * grid[c * M3 + row + idx[2][k]];
                }
            }
        for (int c = 0; c < C; ++c) out[(size_t)r * C + c] = acc[c];
    }
}

/* ---- real-space pair sum ---- */
static const double RS2 = 0.70710678118654752440, RS6 = 0.40824829046386301637;

/* S (3x3 symmetric traceless) from its 5 coordinates in the orthonormal basis e1..e5 (reading R9) */
static void to_tensor(const double *s, double T[3][3]) {
    T[0][0] = s[0] * RS2 - s[1] * RS6; T[1][1] = -s[0] * RS2 - s[1] * RS6; T[2][2] = 2.0 * s[1] * RS6;
    T[0][1] = T[1][0] = s[2] * RS2; T[0][2] = T[2][0] = s[3] * RS2; T[1][2] = T[2][1] = s[4] * RS2;
}
static void to_coords(double T[3][3], double *s) {
    s[0] = (T[0][0] - T[1][1]) * RS2; s[1] = (2.0 * T[2][2] - T[0][0] - T[1][1]) * RS6;
    s[2] = (T[0][1] + T[1][0]) * RS2; s[3] = (T[0][2] + T[2][0]) * RS2; s[4] = (T[1][2] + T[2][1]) * RS2;
}

/* free-space closed forms, units of 1/(6 pi eta a): F1 F2 G1 G2 Z0 Z2 Z4 */
static void free_space(double r, double a, double f[7]) {
    const double p = r / a;
    if (p > 2.0) {
        const double p2 = p * p, p3 = p2 * p, p4 = p2 * p2, p5 = p4 * p;
        f[0] = 3 / (4 * p) + 1 / (2 * p3); f[1] = 3 / (2 * p) - 1 / p3;
        f[2] = 3 * (5 * p2 + 8) / (20 * p4); f[3] = -3 * (5 * p2 - 8) / (20 * p4);
        f[4] = 0; f[5] = 9 / (2 * p3); f[6] = 9 * (5 * p2 - 14) / (4 * p5);
    } else {
        f[0] = 1 - 9 * p / 32; f[1] = 1 - 3 * p / 16;
        f[2] = 3 * p * (64 - 25 * p) / 320; f[3] = 3 * p * (5 * p - 16) / 320;
        f[4] = 9 * (p - 2) * (p - 2) * (p + 4) / 32; f[5] = -9 * p * (p * p - 6) / 64; f[6] = 9 * p * (p * p + 8) / 512;
    }
    f[2] /= a; f[3] /= a; f[4] /= a * a; f[5] /= a * a; f[6] /= a * a;
}

/* [U;E]_rows = M_r [F;S], sum over all beta != alpha with minimum-image |x_alpha - x_beta| < rcut (rcut <= L/2) plus the
 * self term.  x [N][3] wrapped into [0,L); F [N][3]; S5 [N][5]; wtab [nt][7] = the Gaussian-damped wave integrals W_X at
 * r_i = i*dr (smooth; linear interpolation), so that R_X(r) = Free_X(r) - W_X(r); w0[7] = W_X(0); pref = 1/(6 pi eta a).
 * Linked cells of edge >= rcut; with fewer than 3 cells per side every cell is visited once. */
void ref_pairs(int N, const double *x, const double *F, const double *S5, double L, double a, double rcut, double pref,
               const double *wtab, int nt, double dr, int nrows, const long *rows, double *U, double *E) {
    int nc = (int)floor(L / rcut);
    if (nc < 1) nc = 1;
    const double cell_inv = nc / L;
    const int ncell = nc * nc * nc;
    int *start = (int *)calloc((size_t)ncell + 1, sizeof(int)), *fill = (int *)calloc((size_t)ncell, sizeof(int));
    int *cell_of = (int *)malloc(sizeof(int) * (size_t)N), *order = (int *)malloc(sizeof(int) * (size_t)N);
    for (int i = 0; i < N; ++i) {
        int c[3];
        for (int d = 0; d < 3; ++d) { c[d] = (int)(x[3 * (size_t)i + d] * cell_inv); if (c[d] >= nc) c[d] = nc - 1; if (c[d] < 0) c[d] = 0; }
        cell_of[i] = (c[0] * nc + c[1]) * nc + c[2];
        start[cell_of[i] + 1]++;
    }
    for (int c = 0; c < ncell; ++c) start[c + 1] += start[c];
    for (int i = 0; i < N; ++i) order[start[cell_of[i]] + fill[cell_of[i]]++] = i;
    const int span = nc >= 3 ? 3 : nc;
    const double rc2 = rcut * rcut;
#pragma omp parallel for schedule(dynamic, 64)
    for (int r = 0; r < nrows; ++r) {
        const long al = rows[r];
        const double *xa = x + 3 * (size_t)al;
        double u[3] = {0, 0, 0}, e[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
        const int ca = cell_of[al], cz = ca % nc, cy = (ca / nc) % nc, cx = ca / (nc * nc);
        for (int ix = 0; ix < span; ++ix) for (int iy = 0; iy < span; ++iy) for (int iz = 0; iz < span; ++iz) {
            const int bx = nc >= 3 ? (cx + ix - 1 + nc) % nc : ix, by = nc >= 3 ? (cy + iy - 1 + nc) % nc : iy,
                      bz = nc >= 3 ? (cz + iz - 1 + nc) % nc : iz;
            const int cb = (bx * nc + by) * nc + bz;
            for (int p = start[cb]; p < start[cb + 1]; ++p) {
                const int be = order[p];
                if (be == al) continue;
                double d[3], r2 = 0;
                for (int k = 0; k < 3; ++k) { d[k] = xa[k] - x[3 * (size_t)be + k]; d[k] -= L * rint(d[k] / L); r2 += d[k] * d[k]; }
                if (!(r2 < rc2)) continue;
                const double rr = sqrt(r2), rh[3] = {d[0] / rr, d[1] / rr, d[2] / rr};
                double R[7], fs[7];
                free_space(rr, a, fs);
                const double tt = rr / dr;
                int it = (int)tt; if (it > nt - 2) it = nt - 2;
                const double w1 = tt - it, w0 = 1.0 - w1;
                for (int m = 0; m < 7; ++m) R[m] = fs[m] - (w0 * wtab[7 * (size_t)it + m] + w1 * wtab[7 * (size_t)(it + 1) + m]);
                const double j1x = (R[4] + R[5]) / 3, j3x = (R[5] + R[6]) / 7, j2xx = (j1x + j3x) / 5;
                const double Aa = j1x - 2 * j2xx, Bb = 2 * j3x - R[5] / 2, Cc = j3x, Dd = -R[6];
                const double Ga = R[2] + R[3], Gb = R[2] + 4 * R[3];
                const double *Fb = F + 3 * (size_t)be;
                double S[3][3], t[3], f = 0, q = 0;
                to_tensor(S5 + 5 * (size_t)be, S);
                for (int i = 0; i < 3; ++i) { f += rh[i] * Fb[i]; t[i] = S[i][0] * rh[0] + S[i][1] * rh[1] + S[i][2] * rh[2]; }
                for (int i = 0; i < 3; ++i) q += rh[i] * t[i];
                for (int i = 0; i < 3; ++i) u[i] += R[0] * (Fb[i] - rh[i] * f) + R[1] * rh[i] * f + Ga * t[i] - Gb * rh[i] * q;
                for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
                    e[i][j] += -(Ga * 0.5 * (Fb[i] * rh[j] + rh[i] * Fb[j]) + R[3] * f * (i == j) - Gb * f * rh[i] * rh[j])
                             + Aa * S[i][j] + Bb * (rh[i] * t[j] + t[i] * rh[j]) + Cc * q * (i == j) + Dd * q * rh[i] * rh[j];
            }
        }
        /* self term: R_F1(0) F + (R_Z0(0)/5) S  (Eqs. A4, A12) */
        double fs0[7];
        free_space(0.0, a, fs0);
        const double rf1 = fs0[0] - wtab[0], rz0 = fs0[4] - wtab[4];
        double s5[5];
        to_coords(e, s5);
        for (int i = 0; i < 3; ++i) U[3 * (size_t)r + i] = pref * (u[i] + rf1 * F[3 * (size_t)al + i]);
        for (int m = 0; m < 5; ++m) E[5 * (size_t)r + m] = pref * (s5[m] + rz0 / 5.0 * S5[5 * (size_t)al + m]);
    }
    free(start); free(fill); free(cell_of); free(order);
}

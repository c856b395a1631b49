// Real-space table generator (host, fp64 -> fp32).  Product code: shares nothing with oracle/.
//
// The seven scalar functions of M^(r) (Eqs. 25-27) are evaluated as
//     R_X(r) = Free_X(r) - W_X(r; xi)
// with Free_X the free-space Rotne-Prager-type closed forms and W_X the inverse Fourier transform of the
// wave-space summands of Eqs. (21)-(24), reduced to 1-D integrals over spherical Bessel
// functions and done by panelled Gauss-Legendre quadrature (Appendix A of the paper is garbled in
// the extraction and is not used).  The table stores the combinations the pair kernel needs, already multiplied
// by 1/(6 pi eta a):  (F1, F2, G1+G2, G1+4G2, A, B, D, 0)  at r_i = i * dr, i = 0..ntab-1, dr = rcut/(ntab-2).
#include <algorithm>
#include <cmath>
#include <vector>
#include "pse_internal.h"

namespace {

// spherical Bessel j_0..j_4 at x >= 0
void sph_bessel(double x, double j[5]) {
    if (x < 1.0) {                              // ascending series, 10 terms: error < 1e-17 for x < 1
        double x2 = x * x, xl = 1.0, dfact = 1.0;
        for (int l = 0; l <= 4; ++l) {
            dfact *= (2 * l + 1);
            double term = 1.0, sum = 1.0;
            for (int m = 1; m <= 10; ++m) {
                term *= -x2 / (2.0 * m * (2.0 * m + 2 * l + 1));
                sum += term;
            }
            j[l] = xl / dfact * sum;
            xl *= x;
        }
        return;
    }
    double s = std::sin(x), c = std::cos(x);
    j[0] = s / x;
    j[1] = s / (x * x) - c / x;
    for (int l = 1; l < 4; ++l) j[l + 1] = (2 * l + 1) / x * j[l] - j[l - 1];
}

void gauss_legendre(int n, std::vector<double> &x, std::vector<double> &w) {
    x.resize(n); w.resize(n);
    for (int i = 0; i < n; ++i) {
        double z = std::cos(M_PI * (i + 0.75) / (n + 0.5)), pp = 0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1, p2 = 0;
            for (int k = 1; k <= n; ++k) { double p3 = p2; p2 = p1; p1 = ((2 * k - 1) * z * p2 - (k - 1) * p3) / k; }
            pp = n * (z * p1 - p2) / (z * z - 1);
            double dz = p1 / pp; z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        x[i] = z; w[i] = 2.0 / ((1 - z * z) * pp * pp);
    }
}

void free_space(double r, double a, double f[7]) {   // F1 F2 G1 G2 Z0 Z2 Z4
    double p = r / a;
    if (p > 2.0) {
        double p2 = p * p, p3 = p2 * p, p4 = p2 * p2, p5 = p4 * p;
        f[0] = 3 / (4 * p) + 1 / (2 * p3);          f[1] = 3 / (2 * p) - 1 / p3;
        f[2] = 3 * (5 * p2 + 8) / (20 * p4);        f[3] = -3 * (5 * p2 - 8) / (20 * p4);
        f[4] = 0;  f[5] = 9 / (2 * p3);             f[6] = 9 * (5 * p2 - 14) / (4 * p5);
    } else {
        f[0] = 1 - 9 * p / 32;                      f[1] = 1 - 3 * p / 16;
        f[2] = 3 * p * (64 - 25 * p) / 320;         f[3] = 3 * p * (5 * p - 16) / 320;
        f[4] = 9 * (p - 2) * (p - 2) * (p + 4) / 32;
        f[5] = -9 * p * (p * p - 6) / 64;           f[6] = 9 * p * (p * p + 8) / 512;
    }
    f[2] /= a; f[3] /= a; f[4] /= a * a; f[5] /= a * a; f[6] /= a * a;
}

}  // namespace

// R_X(r_i) = Free_X - W_X at the table nodes r_i = i dr, X = F1 F2 G1 G2 Z0 Z2 Z4, in units of 1/(6 pi eta a)
static void real_space_nodes(double a, double xi, double rcut, int ntab, std::vector<double> &R, double *dr_out) {
    const double dr = rcut / (ntab - 2);         // node ntab-2 sits at rcut; one guard node beyond
    const double kmax = 2.0 * xi * std::sqrt(48.0);
    const int npanel = (int)std::ceil(kmax * (rcut + dr + 2 * a) / M_PI) + 8;
    std::vector<double> gx, gw;
    gauss_legendre(16, gx, gw);
    const int nq = npanel * 16;
    std::vector<double> k(nq), c00(nq), c01(nq), c11(nq);
    for (int p = 0; p < npanel; ++p)
        for (int i = 0; i < 16; ++i) {
            double lo = kmax * p / npanel, hi = kmax * (p + 1) / npanel;
            double kk = 0.5 * (lo + hi) + 0.5 * (hi - lo) * gx[i], w = 0.5 * (hi - lo) * gw[i];
            double q = kk * kk / (4 * xi * xi), H = (1 + q) * std::exp(-q);        // Eq. (28)
            double j[5]; sph_bessel(kk * a, j);
            double s0 = j[0], s1 = (kk * a > 1e-8) ? 3 * j[1] / (kk * a) : 1.0;       // shape factors
            int n = p * 16 + i;
            k[n] = kk; c00[n] = w * H * s0 * s0; c01[n] = w * H * kk * s0 * s1; c11[n] = w * H * kk * kk * s1 * s1;
        }
    const double pref = 3.0 * a / M_PI;
    R.assign((size_t)ntab * 7, 0.0);
    for (int i = 0; i < ntab; ++i) {
        double r = i * dr, W[7] = {0, 0, 0, 0, 0, 0, 0};
        for (int n = 0; n < nq; ++n) {
            double x = k[n] * r, j[5]; sph_bessel(x, j);
            double j1x = (x > 1e-12) ? j[1] / x : 1.0 / 3.0, j2x = (x > 1e-12) ? j[2] / x : 0.0;
            W[0] += c00[n] * (j[0] - j1x);   W[1] += c00[n] * 2 * j1x;
            W[2] += c01[n] * (j[1] - j2x);   W[3] -= c01[n] * j2x;
            W[4] += c11[n] * j[0];           W[5] += c11[n] * j[2];          W[6] += c11[n] * j[4];
        }
        double f[7]; free_space(r, a, f);
        for (int m = 0; m < 7; ++m) R[(size_t)i * 7 + m] = f[m] - pref * W[m];
    }
    *dr_out = dr;
}

void pse_build_table(double a, double eta, double xi, double rcut, int ntab, std::vector<float> &tab, double *dr_out) {
    std::vector<double> Rn;
    real_space_nodes(a, xi, rcut, ntab, Rn, dr_out);
    const double unit = 1.0 / (6.0 * M_PI * eta * a);
    tab.assign((size_t)ntab * 8, 0.f);
    for (int i = 0; i < ntab; ++i) {
        const double *R = &Rn[(size_t)i * 7];
        double j1x = (R[4] + R[5]) / 3, j3x = (R[5] + R[6]) / 7, j2xx = (j1x + j3x) / 5;
        float *t = &tab[(size_t)i * 8];
        t[0] = (float)(unit * R[0]);                 t[1] = (float)(unit * R[1]);
        t[2] = (float)(unit * (R[2] + R[3]));        t[3] = (float)(unit * (R[2] + 4 * R[3]));
        t[4] = (float)(unit * (j1x - 2 * j2xx));     t[5] = (float)(unit * (2 * j3x - R[5] / 2));
        t[6] = (float)(unit * (-R[6]));              t[7] = 0.f;
    }
}

// Scalar functions of the rotational couplings (torque in, angular velocity out; reading R21) at the same nodes:
// (T/2, Z0/6, Z2/4, 0) with T = G1 - G2, times 1/(6 pi eta a).  The antisymmetric part of Eq. (26) contracts to G1 - G2, and the
// L / Omega couplings carry the weight k^2 s1^2 of Z0, Z2: no new integral.
void pse_build_rot_table(double a, double eta, double xi, double rcut, int ntab, std::vector<float> &tab) {
    std::vector<double> Rn;
    double dr;
    real_space_nodes(a, xi, rcut, ntab, Rn, &dr);
    const double unit = 1.0 / (6.0 * M_PI * eta * a);
    tab.assign((size_t)ntab * 4, 0.f);
    for (int i = 0; i < ntab; ++i) {
        const double *R = &Rn[(size_t)i * 7];
        float *t = &tab[(size_t)i * 4];
        t[0] = (float)(unit * 0.5 * (R[2] - R[3])); t[1] = (float)(unit * R[4] / 6.0); t[2] = (float)(unit * R[5] / 4.0); t[3] = 0.f;
    }
}

// ---- spreading / interpolation window and its transform ----
// kappa(k_n) = int_{-P/2}^{P/2} w(t) cos(2 pi n t / M) dt  (t in grid units) is the continuous transform of the 1-D
// window that the P-point sums approximate; the scale kernel multiplies by 1/kappa per dimension, once for spreading
// and once for interpolation (R4).  dec[i] = 1/kappa for FFT index i (signed wave number n = i or i - M).
void pse_window_table(int kind, int P, double wa, double wb, int M, std::vector<float> &dec) {
    std::vector<double> gx, gw;
    gauss_legendre(32, gx, gw);
    const int npanel = 4 * P;                              // panels of width 1/4 grid spacing, 32 nodes each
    dec.assign(M, 0.f);
    for (int i = 0; i < M; ++i) {
        const int n = i < (M + 1) / 2 ? i : i - M;
        const double kh = 2.0 * M_PI * n / M;
        double kap = 0;
        for (int p = 0; p < npanel; ++p) {
            const double lo = -0.5 * P + (double)P * p / npanel, hi = -0.5 * P + (double)P * (p + 1) / npanel;
            for (int q = 0; q < 32; ++q) {
                const double t = 0.5 * (lo + hi) + 0.5 * (hi - lo) * gx[q];
                const double arg = kind ? wb * (std::sqrt(std::max(1.0 - wa * t * t, 0.0)) - 1.0) : -wa * t * t;
                kap += 0.5 * (hi - lo) * gw[q] * std::exp(arg) * std::cos(kh * t);
            }
        }
        dec[i] = (float)(1.0 / kap);
    }
}

// shape parameter of the exponential-of-semicircle window: beta = 2.2 P (calibrated against the oracle, R3/R6)
double pse_es_beta(int P) { return 2.2 * P; }

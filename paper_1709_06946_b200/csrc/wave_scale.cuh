// k-space operator of the wave-space sum (used by the scaling kernels of wavespace.cu).  Eqs. (21)-(24), (41).
#pragma once
#include <cmath>
#include "pse_internal.h"

namespace {

constexpr float WS_RS2 = 0.70710678118654752f, WS_RS6 = 0.40824829046386302f;

struct ScaleParams {
    int M, Mh;
    int Mc, Mch;                                   // Brownian pass on the finer grid: the (coarser) product grid the noise buffer is laid out on
    float two_pi_over_L, a, inv4xi2, c_mv, c_br, inv_eta;
    const float *dec;                              // [M] 1/kappa(k_n): inverse 1-D window transform per FFT index
    int mode;                                      // PSE_IN_F | PSE_IN_S | PSE_OUT_U | PSE_OUT_E: which planes are read / written
    const Lat *lat;                                // k = (2 pi/L) A^-T n: kx = i11 nx, ky = i22 ny + i12 nx (entries of A^-1; 1, 0, 1 on the cube), read from
                                                   // device memory so that a captured step stays valid while the strain advances
};

// s0 = sin x / x and s1 = 3 (sin x - x cos x)/x^3 (series below 0.5: cancellation) from one sincosf, x > 0
__device__ __forceinline__ void shape_factors(float x, float &s0, float &s1) {
    float s, c; sincosf(x, &s, &c);
    const float ix = 1.f / x;
    s0 = s * ix;
    if (x < 0.5f) { const float x2 = x * x; s1 = 1.f - x2 * (0.1f - x2 * (1.f / 280.f - x2 * (1.f / 15120.f))); }
    else s1 = 3.f * (s - x * c) * (ix * ix * ix);
}

// Wave vector of half-spectrum entry (ix,iy,iz); returns false for k = 0 and Nyquist modes (weight set to zero in
// both the product and the Brownian factor, reading R8).
__device__ __forceinline__ bool mode_k(const ScaleParams &sp, int ix, int iy, int iz, float &kx, float &ky, float &kz) {
    const int M = sp.M, half = (M + 1) / 2;
    const int nx = ix < half ? ix : ix - M, ny = iy < half ? iy : iy - M, nz = iz;
    const bool nyq = !(M & 1) && (ix == M / 2 || iy == M / 2 || iz == M / 2);
    const float ki11 = __ldg(&sp.lat->i11), ki12 = __ldg(&sp.lat->i12), ki22 = __ldg(&sp.lat->i22);
    kx = sp.two_pi_over_L * (ki11 * (float)nx); ky = sp.two_pi_over_L * (ki22 * (float)ny + ki12 * (float)nx); kz = sp.two_pi_over_L * (float)nz;
    return !(nyq || (nx == 0 && ny == 0 && nz == 0));
}

// Given uh (3 complex, already carrying B or sqrt(B) and the projector), write the 8 outputs of P^H (Eq. 41):
//   Uh = s0 uh ;  Eh^q = i s1 (e^q k).uh
__device__ __forceinline__ void write_outputs(float2 *spec, size_t stride, size_t o, float s0, float s1,
                                              float kx, float ky, float kz, float2 ux, float2 uy, float2 uz, int mode) {
    if (mode & PSE_OUT_U) {
        spec[o] = make_float2(s0 * ux.x, s0 * ux.y);
        spec[stride + o] = make_float2(s0 * uy.x, s0 * uy.y);
        spec[2 * stride + o] = make_float2(s0 * uz.x, s0 * uz.y);
    }
    if (!(mode & PSE_OUT_E)) return;
    // i*s1*z = s1 * (-z.im, z.re)
    float2 pxx = make_float2(kx * ux.x, kx * ux.y), pyy = make_float2(ky * uy.x, ky * uy.y), pzz = make_float2(kz * uz.x, kz * uz.y);
    float2 d1 = make_float2((pxx.x - pyy.x) * WS_RS2, (pxx.y - pyy.y) * WS_RS2);
    float2 d2 = make_float2((2.f * pzz.x - pxx.x - pyy.x) * WS_RS6, (2.f * pzz.y - pxx.y - pyy.y) * WS_RS6);
    float2 d3 = make_float2((kx * uy.x + ky * ux.x) * WS_RS2, (kx * uy.y + ky * ux.y) * WS_RS2);
    float2 d4 = make_float2((kx * uz.x + kz * ux.x) * WS_RS2, (kx * uz.y + kz * ux.y) * WS_RS2);
    float2 d5 = make_float2((ky * uz.x + kz * uy.x) * WS_RS2, (ky * uz.y + kz * uy.y) * WS_RS2);
    spec[3 * stride + o] = make_float2(-s1 * d1.y, s1 * d1.x);
    spec[4 * stride + o] = make_float2(-s1 * d2.y, s1 * d2.x);
    spec[5 * stride + o] = make_float2(-s1 * d3.y, s1 * d3.x);
    spec[6 * stride + o] = make_float2(-s1 * d4.y, s1 * d4.x);
    spec[7 * stride + o] = make_float2(-s1 * d5.y, s1 * d5.x);
}

// a5 at one mode: fh = s0 Fh - i s1 (Sh.k);  uh = Bt(k) (I - kh kh) fh  with
// Bt = c_mv (1+k^2/4xi^2) exp(-k^2/4xi^2)/(eta k^2) / kappa(k)^2.  Inputs are read from in[c*in_stride + oi] (component c
// present in sp.mode), outputs written to out[c*out_stride + oo]; all reads precede the writes, so in == out is fine.
__device__ __forceinline__ void scale_point(const ScaleParams &sp, int ix, int iy, int iz, const float2 *in, size_t in_stride, size_t oi,
                                            float2 *out, size_t out_stride, size_t oo) {
    float kx, ky, kz;
    const float2 zero = make_float2(0.f, 0.f);
    if (!mode_k(sp, ix, iy, iz, kx, ky, kz)) {
#pragma unroll
        for (int c = 0; c < 8; ++c)
            if (sp.mode & (c < 3 ? PSE_OUT_U : PSE_OUT_E)) out[c * out_stride + oo] = zero;
        return;
    }
    const float k2 = kx * kx + ky * ky + kz * kz, kn = sqrtf(k2), ka = kn * sp.a;
    float s0, s1;
    shape_factors(ka, s0, s1);
    const float q = k2 * sp.inv4xi2;
    const float dw = __ldg(sp.dec + ix) * __ldg(sp.dec + iy) * __ldg(sp.dec + iz);            // one window undone for spreading,
    const float Bt = sp.c_mv * sp.inv_eta * (1.f + q) * __expf(-q) / k2 * dw * dw;          // one for interpolation
    float2 F[3], S[5];
#pragma unroll
    for (int c = 0; c < 3; ++c) F[c] = (sp.mode & PSE_IN_F) ? in[c * in_stride + oi] : zero;
#pragma unroll
    for (int c = 0; c < 5; ++c) S[c] = (sp.mode & PSE_IN_S) ? in[(3 + c) * in_stride + oi] : zero;
    // (S.k)_i from the 5 coordinates
    float2 sk[3];
#pragma unroll
    for (int ri = 0; ri < 2; ++ri) {
        float s1c = ri ? S[0].y : S[0].x, s2c = ri ? S[1].y : S[1].x, s3c = ri ? S[2].y : S[2].x, s4c = ri ? S[3].y : S[3].x,
              s5c = ri ? S[4].y : S[4].x;
        float sxx = s1c * WS_RS2 - s2c * WS_RS6, syy = -s1c * WS_RS2 - s2c * WS_RS6, szz = 2.f * s2c * WS_RS6;
        float sxy = s3c * WS_RS2, sxz = s4c * WS_RS2, syz = s5c * WS_RS2;
        float vx = sxx * kx + sxy * ky + sxz * kz, vy = sxy * kx + syy * ky + syz * kz, vz = sxz * kx + syz * ky + szz * kz;
        if (ri) { sk[0].y = vx; sk[1].y = vy; sk[2].y = vz; } else { sk[0].x = vx; sk[1].x = vy; sk[2].x = vz; }
    }
    // fh = s0 F - i s1 sk = s0 F + s1 (sk.im, -sk.re)
    float2 f[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) f[c] = make_float2(s0 * F[c].x + s1 * sk[c].y, s0 * F[c].y - s1 * sk[c].x);
    const float ik2 = 1.f / k2;
    const float2 kf = make_float2((kx * f[0].x + ky * f[1].x + kz * f[2].x) * ik2, (kx * f[0].y + ky * f[1].y + kz * f[2].y) * ik2);
    const float2 ux = make_float2(Bt * (f[0].x - kx * kf.x), Bt * (f[0].y - kx * kf.y));
    const float2 uy = make_float2(Bt * (f[1].x - ky * kf.x), Bt * (f[1].y - ky * kf.y));
    const float2 uz = make_float2(Bt * (f[2].x - kz * kf.x), Bt * (f[2].y - kz * kf.y));
    write_outputs(out, out_stride, oo, s0, s1, kx, ky, kz, ux, uy, uz, sp.mode);
}

inline ScaleParams make_scale_params(const pse_ctx *c, int mode = PSE_MODE_ALL) {
    ScaleParams sp;
    sp.mode = mode;
    sp.M = c->M; sp.Mh = c->Mh; sp.Mc = c->M; sp.Mch = c->Mh;
    sp.two_pi_over_L = (float)(2.0 * M_PI / c->L); sp.a = (float)c->a;
    sp.inv4xi2 = (float)(1.0 / (4.0 * c->xi * c->xi)); sp.dec = c->d_dec;
    const double V = c->L * c->L * c->L;
    sp.c_mv = (float)(1.0 / V); sp.c_br = (float)(1.0 / std::sqrt(V));
    sp.inv_eta = (float)(1.0 / c->eta);
    sp.lat = c->d_lat;
    return sp;
}

}  // namespace

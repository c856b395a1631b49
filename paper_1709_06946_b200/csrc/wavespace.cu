// Wave-space half of the product: M_w = sigma Q^T F^H P^H B P F Q (Eq. 42) and the Brownian factor
// M_w^{1/2} = sigma^{1/2} Q^T F^H P^H B^{1/2} (Eq. 75).  Steps a3-a7 of SURVEY.md §8(a).
//
// Grid layout: 8 planar real grids [c][ix][iy][iz] (iz fastest), grid point n at n*h; half spectrum
// [c][ix][iy][iz<=M/2].  c = (Fx,Fy,Fz,S1..S5) going in, (Ux,Uy,Uz,E1..E5) coming out.
// Gaussian (R3-R5): K(r) = (2 xi^2/(pi eta_g))^{3/2} exp(-2 xi^2 r^2/eta_g) with
// eta_g = (h P xi/m)^2, m = sqrt(pi P), so on the grid K ~ exp(-(2 pi/P) t^2), t = distance in grid units: the
// weights depend on P only.  All constant prefactors (both Gaussians' normalisation, h^3 of the two quadratures,
// 1/V) are folded into the scale kernel: (2/P)^3/V for the product, (2/P)^{3/2}/sqrt(V) for the Brownian factor.
//
// Spread is written in GATHER form (not the paper's per-particle atomics): one CTA owns an 8^3 tile
// of grid points, one thread per point with the 8 components in registers; it walks the particles binned in the
// tiles whose supports can reach it, with separable weights staged in shared memory.  No atomics, no memset,
// each grid value is written exactly once with full-sector coalesced stores, and the summation order is fixed.
#include "pse_internal.h"

namespace {

constexpr int T = PSE_TILE;
constexpr float RS2 = 0.70710678118654752f, RS6 = 0.40824829046386302f;
constexpr float TWO_PI = 6.283185307179586f;

// support base (unwrapped, may be negative) and grid coordinate g = x/h   (reading R5)
__device__ __forceinline__ int support_base(float g, int P) {
    return (P & 1) ? (int)rintf(g) - (P - 1) / 2 : (int)floorf(g) - P / 2 + 1;
}
__device__ __forceinline__ int pmod(int i, int M) { int r = i % M; return r < 0 ? r + M : r; }

__global__ void tile_of_particles(const float4 *pos, int N, float inv_h, int M, int P, int nt, int *tile_of, int *tile_count) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    float4 p = pos[s];
    int tx = pmod(support_base(p.x * inv_h, P), M) / T, ty = pmod(support_base(p.y * inv_h, P), M) / T,
        tz = pmod(support_base(p.z * inv_h, P), M) / T;
    int t = (tx * nt + ty) * nt + tz;
    tile_of[s] = t;
    atomicAdd(&tile_count[t], 1);
}

__global__ void scatter_to_tiles(const int *tile_of, int N, const int *tile_start, int *tile_fill, int *tile_list) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    int t = tile_of[s];
    tile_list[tile_start[t] + atomicAdd(&tile_fill[t], 1)] = s;
}

__global__ void sort_within_tiles(const int *tile_start, int ntile, int *tile_list) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntile) return;
    int lo = tile_start[t], hi = tile_start[t + 1];
    for (int i = lo + 1; i < hi; ++i) {
        int v = tile_list[i], j = i - 1;
        while (j >= lo && tile_list[j] > v) { tile_list[j + 1] = tile_list[j]; --j; }
        tile_list[j + 1] = v;
    }
}

// Tiles (along one axis) whose particles' supports can reach tile t: bases in [t*T-(P-1), t*T+T-1] mod M.
__device__ int reach_tiles(int t, int M, int P, int nt, int *list) {
    int n = 0;
    for (int j = P - 1; j >= 0; --j) {
        int tb = pmod(t * T - j, M) / T;
        bool seen = false;
        for (int q = 0; q < n; ++q) seen |= (list[q] == tb);
        if (!seen && n < 4) list[n++] = tb;
    }
    (void)nt;
    return n;
}

constexpr int SPREAD_BATCH = 64;

__global__ void __launch_bounds__(512)
spread_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ in, const int *__restrict__ tile_start,
              const int *__restrict__ tile_list, float *__restrict__ grid, int M, int P, int nt, float inv_h, float wexp) {
    __shared__ float4 q[SPREAD_BATCH][2];
    __shared__ float W[SPREAD_BATCH][3][T];
    __shared__ float gco[SPREAD_BATCH][3];
    __shared__ int gbase[SPREAD_BATCH][3];
    __shared__ int active[SPREAD_BATCH];
    __shared__ int bin_lo[64], bin_cum[65], nbins_s;
    const int tid = threadIdx.x, a = tid >> 6, b = (tid >> 3) & 7, cc = tid & 7;
    const int t = blockIdx.x, t0 = t / (nt * nt), t1 = (t / nt) % nt, t2 = t % nt;
    const int g0[3] = {t0 * T, t1 * T, t2 * T};
    if (tid == 0) {
        int lx[4], ly[4], lz[4];
        int nx = reach_tiles(t0, M, P, nt, lx), ny = reach_tiles(t1, M, P, nt, ly), nz = reach_tiles(t2, M, P, nt, lz);
        int n = 0, cum = 0;
        for (int i = 0; i < nx; ++i) for (int j = 0; j < ny; ++j) for (int k = 0; k < nz; ++k) {
            int tb = (lx[i] * nt + ly[j]) * nt + lz[k];
            bin_lo[n] = tile_start[tb]; bin_cum[n] = cum; cum += tile_start[tb + 1] - tile_start[tb]; ++n;
        }
        bin_cum[n] = cum; nbins_s = n;
    }
    __syncthreads();
    const int nbins = nbins_s, total = bin_cum[nbins];
    float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int lo = 0; lo < total; lo += SPREAD_BATCH) {
        const int nb = min(SPREAD_BATCH, total - lo);
        if (tid < nb) {
            int ci = lo + tid, k = 0;
            while (bin_cum[k + 1] <= ci) ++k;
            int s = tile_list[bin_lo[k] + ci - bin_cum[k]];
            float4 p = pos[s];
            q[tid][0] = in[2 * s]; q[tid][1] = in[2 * s + 1];
            float g[3] = {p.x * inv_h, p.y * inv_h, p.z * inv_h};
            for (int d = 0; d < 3; ++d) { gco[tid][d] = g[d]; gbase[tid][d] = support_base(g[d], P); }
        }
        __syncthreads();
        for (int e = tid; e < nb * 3 * T; e += blockDim.x) {
            int p = e / (3 * T), d = (e / T) % 3, i = e % T;
            int gp = g0[d] + i, base = gbase[p][d];
            int o = pmod(gp - base, M);
            float tt = (float)(base + o) - gco[p][d];
            W[p][d][i] = (o < P && gp < M) ? __expf(-wexp * tt * tt) : 0.f;
        }
        __syncthreads();
        if (tid < nb) {
            bool any[3] = {false, false, false};
            for (int d = 0; d < 3; ++d) for (int i = 0; i < T; ++i) any[d] |= (W[tid][d][i] != 0.f);
            active[tid] = any[0] && any[1] && any[2];
        }
        __syncthreads();
        for (int p = 0; p < nb; ++p) {
            if (!active[p]) continue;
            const float wx = W[p][0][a];
            if (wx == 0.f) continue;                                  // warp-uniform (a is fixed within a warp)
            const float w = wx * W[p][1][b] * W[p][2][cc];
            const float4 q0 = q[p][0], q1 = q[p][1];
            acc[0] += w * q0.x; acc[1] += w * q0.y; acc[2] += w * q0.z; acc[3] += w * q0.w;
            acc[4] += w * q1.x; acc[5] += w * q1.y; acc[6] += w * q1.z; acc[7] += w * q1.w;
        }
        __syncthreads();
    }
    const int gx = g0[0] + a, gy = g0[1] + b, gz = g0[2] + cc;
    if (gx < M && gy < M && gz < M) {
        const size_t M3 = (size_t)M * M * M, o = ((size_t)gx * M + gy) * M + gz;
#pragma unroll
        for (int c = 0; c < 8; ++c) grid[c * M3 + o] = acc[c];
    }
}

// Interpolation (a7): warp per particle (visited in tile order for L1/L2 locality), lanes over the P^3 support.
__global__ void __launch_bounds__(256)
interp_kernel(const float4 *__restrict__ pos, const int *__restrict__ tile_list, const float *__restrict__ grid,
              float4 *__restrict__ out, int N, int M, int P, float inv_h, float wexp, int accumulate) {
    const int wi = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (wi >= N) return;
    const int s = tile_list[wi];
    const float4 p = pos[s];
    const float g[3] = {p.x * inv_h, p.y * inv_h, p.z * inv_h};
    int base[3];
    for (int d = 0; d < 3; ++d) base[d] = support_base(g[d], P);
    float wr[2];
    for (int h = 0; h < 2; ++h) {                       // entry e = d*P + i, e < 3P <= 48
        int e = lane + 32 * h, d = e / P, i = e % P;
        float tt = (d < 3) ? (float)(base[d] + i) - g[d] : 0.f;
        wr[h] = (d < 3) ? __expf(-wexp * tt * tt) : 0.f;
    }
    const size_t M3 = (size_t)M * M * M;
    float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const int P2 = P * P, P3 = P2 * P;
    for (int pt0 = 0; pt0 < P3; pt0 += 32) {
        const int pt = pt0 + lane;
        const bool ok = pt < P3;
        const int ptc = ok ? pt : 0;
        const int i = ptc / P2, j = (ptc / P) % P, k = ptc % P;
        const int ez = 2 * P + k;                          // entries: x at i, y at P+j (< 32 for P <= 16), z at 2P+k
        const float wx = __shfl_sync(0xffffffffu, wr[0], i), wy = __shfl_sync(0xffffffffu, wr[0], P + j);
        const float wz0 = __shfl_sync(0xffffffffu, wr[0], ez & 31), wz1 = __shfl_sync(0xffffffffu, wr[1], ez & 31);
        const float w = ok ? wx * wy * (ez < 32 ? wz0 : wz1) : 0.f;
        const size_t o = ((size_t)pmod(base[0] + i, M) * M + pmod(base[1] + j, M)) * M + pmod(base[2] + k, M);
        if (ok) {
#pragma unroll
            for (int c = 0; c < 8; ++c) acc[c] += w * __ldg(grid + c * M3 + o);
        }
    }
#pragma unroll
    for (int c = 0; c < 8; ++c)
        for (int o = 16; o; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    if (lane == 0) {
        float4 r0 = make_float4(acc[0], acc[1], acc[2], acc[3]), r1 = make_float4(acc[4], acc[5], acc[6], acc[7]);
        if (accumulate) {
            float4 o0 = out[2 * s], o1 = out[2 * s + 1];
            r0.x += o0.x; r0.y += o0.y; r0.z += o0.z; r0.w += o0.w; r1.x += o1.x; r1.y += o1.y; r1.z += o1.z; r1.w += o1.w;
        }
        out[2 * s] = r0; out[2 * s + 1] = r1;
    }
}

struct ScaleParams {
    int M, Mh;
    float two_pi_over_L, a, inv4xi2, one_minus_etag, c_mv, c_br, inv_eta;
};

__device__ __forceinline__ float shape_s1(float x) {     // 3 (sin x - x cos x)/x^3, series below 0.5 (cancellation)
    if (x < 0.5f) { float x2 = x * x; return 1.f - x2 * (0.1f - x2 * (1.f / 280.f - x2 * (1.f / 15120.f))); }
    float s, c; sincosf(x, &s, &c);
    return 3.f * (s - x * c) / (x * x * x);
}

// Wave vector of half-spectrum entry (ix,iy,iz); returns false for k = 0 and Nyquist modes (weight set to zero in
// both the product and the Brownian factor, reading R8).
__device__ __forceinline__ bool mode_k(const ScaleParams &sp, int ix, int iy, int iz, float &kx, float &ky, float &kz) {
    const int M = sp.M, half = (M + 1) / 2;
    const int nx = ix < half ? ix : ix - M, ny = iy < half ? iy : iy - M, nz = iz;
    const bool nyq = !(M & 1) && (ix == M / 2 || iy == M / 2 || iz == M / 2);
    kx = sp.two_pi_over_L * (float)nx; ky = sp.two_pi_over_L * (float)ny; kz = sp.two_pi_over_L * (float)nz;
    return !(nyq || (nx == 0 && ny == 0 && nz == 0));
}

// Given uh (3 complex, already carrying B or sqrt(B) and the projector), write the 8 outputs of P^H (Eq. 41):
//   Uh = s0 uh ;  Eh^q = i s1 (e^q k).uh
__device__ __forceinline__ void write_outputs(cufftComplex *spec, size_t stride, size_t o, float s0, float s1,
                                              float kx, float ky, float kz, float2 ux, float2 uy, float2 uz) {
    spec[o] = make_float2(s0 * ux.x, s0 * ux.y);
    spec[stride + o] = make_float2(s0 * uy.x, s0 * uy.y);
    spec[2 * stride + o] = make_float2(s0 * uz.x, s0 * uz.y);
    // i*s1*z = s1 * (-z.im, z.re)
    float2 pxx = make_float2(kx * ux.x, kx * ux.y), pyy = make_float2(ky * uy.x, ky * uy.y), pzz = make_float2(kz * uz.x, kz * uz.y);
    float2 d1 = make_float2((pxx.x - pyy.x) * RS2, (pxx.y - pyy.y) * RS2);
    float2 d2 = make_float2((2.f * pzz.x - pxx.x - pyy.x) * RS6, (2.f * pzz.y - pxx.y - pyy.y) * RS6);
    float2 d3 = make_float2((kx * uy.x + ky * ux.x) * RS2, (kx * uy.y + ky * ux.y) * RS2);
    float2 d4 = make_float2((kx * uz.x + kz * ux.x) * RS2, (kx * uz.y + kz * ux.y) * RS2);
    float2 d5 = make_float2((ky * uz.x + kz * uy.x) * RS2, (ky * uz.y + kz * uy.y) * RS2);
    spec[3 * stride + o] = make_float2(-s1 * d1.y, s1 * d1.x);
    spec[4 * stride + o] = make_float2(-s1 * d2.y, s1 * d2.x);
    spec[5 * stride + o] = make_float2(-s1 * d3.y, s1 * d3.x);
    spec[6 * stride + o] = make_float2(-s1 * d4.y, s1 * d4.x);
    spec[7 * stride + o] = make_float2(-s1 * d5.y, s1 * d5.x);
}

// a5: fh = s0 Fh - i s1 (Sh.k);  uh = Bt(k) (I - kh kh) fh  with  Bt = c_mv (1+k^2/4xi^2) exp(-(1-eta_g) k^2/4xi^2)/(eta k^2)
__global__ void __launch_bounds__(256) scale_kernel(cufftComplex *spec, ScaleParams sp) {
    const size_t nmode = (size_t)sp.M * sp.M * sp.Mh, o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nmode) return;
    const int iz = (int)(o % sp.Mh), iy = (int)((o / sp.Mh) % sp.M), ix = (int)(o / ((size_t)sp.Mh * sp.M));
    float kx, ky, kz;
    float2 zero = make_float2(0.f, 0.f);
    if (!mode_k(sp, ix, iy, iz, kx, ky, kz)) {
#pragma unroll
        for (int c = 0; c < 8; ++c) spec[c * nmode + o] = zero;
        return;
    }
    const float k2 = kx * kx + ky * ky + kz * kz, kn = sqrtf(k2), ka = kn * sp.a;
    const float s0 = sinf(ka) / ka, s1 = shape_s1(ka);
    const float q = k2 * sp.inv4xi2;
    const float Bt = sp.c_mv * sp.inv_eta * (1.f + q) * __expf(-sp.one_minus_etag * q) / k2;
    float2 F[3], S[5];
#pragma unroll
    for (int c = 0; c < 3; ++c) F[c] = spec[c * nmode + o];
#pragma unroll
    for (int c = 0; c < 5; ++c) S[c] = spec[(3 + c) * nmode + o];
    // (S.k)_i from the 5 coordinates
    float2 sk[3];
#pragma unroll
    for (int ri = 0; ri < 2; ++ri) {
        float s1c = ri ? S[0].y : S[0].x, s2c = ri ? S[1].y : S[1].x, s3c = ri ? S[2].y : S[2].x, s4c = ri ? S[3].y : S[3].x,
              s5c = ri ? S[4].y : S[4].x;
        float sxx = s1c * RS2 - s2c * RS6, syy = -s1c * RS2 - s2c * RS6, szz = 2.f * s2c * RS6;
        float sxy = s3c * RS2, sxz = s4c * RS2, syz = s5c * RS2;
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
    write_outputs(spec, nmode, o, s0, s1, kx, ky, kz, ux, uy, uz);
}

// a5, Brownian flavour (Eq. 75): uh = c_br sqrt((1+k^2/4xi^2)/(eta k^2)) exp(-(1-eta_g) k^2/8xi^2) (I - kh kh) W(k),
// W(k) = (g_re + i g_im)/sqrt2 from the noise buffer; in the plane kz = 0 the non-canonical member of each +-k
// pair takes the conjugate of its partner's entry (reading R8) so that the C2R transform sees a Hermitian field.
__global__ void __launch_bounds__(256) scale_brownian_kernel(cufftComplex *spec, const float2 *__restrict__ noise, ScaleParams sp) {
    const size_t nmode = (size_t)sp.M * sp.M * sp.Mh, o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= nmode) return;
    const int M = sp.M;
    const int iz = (int)(o % sp.Mh), iy = (int)((o / sp.Mh) % M), ix = (int)(o / ((size_t)sp.Mh * M));
    float kx, ky, kz;
    float2 zero = make_float2(0.f, 0.f);
    if (!mode_k(sp, ix, iy, iz, kx, ky, kz)) {
#pragma unroll
        for (int c = 0; c < 8; ++c) spec[c * nmode + o] = zero;
        return;
    }
    const int half = (M + 1) / 2, nx = ix < half ? ix : ix - M, ny = iy < half ? iy : iy - M;
    const bool canon = iz > 0 || ny > 0 || (ny == 0 && nx > 0);
    const size_t src = canon ? o : ((size_t)((M - ix) % M) * M + (size_t)((M - iy) % M)) * sp.Mh;
    const float sgn = canon ? 1.f : -1.f;
    float2 W[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { float2 g = noise[c * nmode + src]; W[c] = make_float2(g.x * RS2, sgn * g.y * RS2); }
    const float k2 = kx * kx + ky * ky + kz * kz, kn = sqrtf(k2), ka = kn * sp.a;
    const float s0 = sinf(ka) / ka, s1 = shape_s1(ka);
    const float q = k2 * sp.inv4xi2;
    const float Bh = sp.c_br * sqrtf(sp.inv_eta * (1.f + q) / k2) * __expf(-0.5f * sp.one_minus_etag * q);
    const float ik2 = 1.f / k2;
    const float2 kw = make_float2((kx * W[0].x + ky * W[1].x + kz * W[2].x) * ik2, (kx * W[0].y + ky * W[1].y + kz * W[2].y) * ik2);
    const float2 ux = make_float2(Bh * (W[0].x - kx * kw.x), Bh * (W[0].y - kx * kw.y));
    const float2 uy = make_float2(Bh * (W[1].x - ky * kw.x), Bh * (W[1].y - ky * kw.y));
    const float2 uz = make_float2(Bh * (W[2].x - kz * kw.x), Bh * (W[2].y - kz * kw.y));
    write_outputs(spec, nmode, o, s0, s1, kx, ky, kz, ux, uy, uz);
}

}  // namespace

pse_status pse_wave_init(pse_ctx *c) {
    const int M = c->M;
    c->Mh = M / 2 + 1;
    c->nt = (M + T - 1) / T; c->ntile = c->nt * c->nt * c->nt;
    const size_t M3 = (size_t)M * M * M, nmode = (size_t)M * M * c->Mh;
    CUDA_TRY(c, cudaMalloc(&c->d_grid, 8 * M3 * sizeof(float)));
    CUDA_TRY(c, cudaMalloc(&c->d_spec, 8 * nmode * sizeof(cufftComplex)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_count, (size_t)(c->ntile + 1) * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_start, (size_t)(c->ntile + 1) * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_fill, (size_t)(c->ntile + 1) * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_of, (size_t)c->N * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_list, (size_t)c->N * sizeof(int)));
    int n[3] = {M, M, M};
    size_t w1 = 0, w2 = 0;
    CUFFT_TRY(c, cufftCreate(&c->plan_r2c)); CUFFT_TRY(c, cufftCreate(&c->plan_c2r)); c->have_plans = true;
    CUFFT_TRY(c, cufftSetAutoAllocation(c->plan_r2c, 0)); CUFFT_TRY(c, cufftSetAutoAllocation(c->plan_c2r, 0));
    CUFFT_TRY(c, cufftMakePlanMany(c->plan_r2c, 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, 8, &w1));
    CUFFT_TRY(c, cufftMakePlanMany(c->plan_c2r, 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, 8, &w2));
    size_t w = w1 > w2 ? w1 : w2;
    if (w) CUDA_TRY(c, cudaMalloc(&c->d_fft_work, w));
    CUFFT_TRY(c, cufftSetWorkArea(c->plan_r2c, c->d_fft_work)); CUFFT_TRY(c, cufftSetWorkArea(c->plan_c2r, c->d_fft_work));
    CUFFT_TRY(c, cufftSetStream(c->plan_r2c, c->stream)); CUFFT_TRY(c, cufftSetStream(c->plan_c2r, c->stream));
    return PSE_OK;
}

void pse_wave_free(pse_ctx *c) {
    if (c->have_plans) { cufftDestroy(c->plan_r2c); cufftDestroy(c->plan_c2r); }
    cudaFree(c->d_grid); cudaFree(c->d_spec); cudaFree(c->d_fft_work);
    cudaFree(c->d_tile_count); cudaFree(c->d_tile_start); cudaFree(c->d_tile_fill); cudaFree(c->d_tile_of); cudaFree(c->d_tile_list);
}

pse_status pse_tile_bins(pse_ctx *c) {
    const int N = c->N, TB = 256, nb = (N + TB - 1) / TB;
    CUDA_TRY(c, cudaMemsetAsync(c->d_tile_count, 0, (size_t)(c->ntile + 1) * sizeof(int), c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->d_tile_fill, 0, (size_t)(c->ntile + 1) * sizeof(int), c->stream));
    tile_of_particles<<<nb, TB, 0, c->stream>>>(c->d_pos, N, (float)(1.0 / c->h), c->M, c->P, c->nt, c->d_tile_of, c->d_tile_count); KERNEL_CHECK(c);
    PSE_TRY(pse_scan_i32(c, c->d_tile_count, c->d_tile_start, (size_t)c->ntile));
    scatter_to_tiles<<<nb, TB, 0, c->stream>>>(c->d_tile_of, N, c->d_tile_start, c->d_tile_fill, c->d_tile_list); KERNEL_CHECK(c);
    sort_within_tiles<<<(c->ntile + 127) / 128, 128, 0, c->stream>>>(c->d_tile_start, c->ntile, c->d_tile_list); KERNEL_CHECK(c);
    return PSE_OK;
}

static ScaleParams make_scale_params(const pse_ctx *c) {
    ScaleParams sp;
    sp.M = c->M; sp.Mh = c->Mh;
    sp.two_pi_over_L = (float)(2.0 * M_PI / c->L); sp.a = (float)c->a;
    sp.inv4xi2 = (float)(1.0 / (4.0 * c->xi * c->xi)); sp.one_minus_etag = (float)(1.0 - c->eta_g);
    const double V = c->L * c->L * c->L, tp = 2.0 / c->P;
    sp.c_mv = (float)(tp * tp * tp / V); sp.c_br = (float)(std::sqrt(tp * tp * tp / V));
    sp.inv_eta = (float)(1.0 / c->eta);
    return sp;
}

static pse_status inverse_and_interpolate(pse_ctx *c, float *d_out, bool accumulate) {
    { ScopedPhase ph(c, PSE_T_FFT_INV); CUFFT_TRY(c, cufftExecC2R(c->plan_c2r, c->d_spec, c->d_grid)); c->launches++; }
    ScopedPhase ph(c, PSE_T_INTERP);
    const int TB = 256;
    interp_kernel<<<(unsigned)(((size_t)c->N * 32 + TB - 1) / TB), TB, 0, c->stream>>>(
        c->d_pos, c->d_tile_list, c->d_grid, reinterpret_cast<float4 *>(d_out), c->N, c->M, c->P, (float)(1.0 / c->h),
        (float)(2.0 * M_PI / c->P), accumulate ? 1 : 0);
    KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_wave_apply(pse_ctx *c, const float *d_in, float *d_out, bool accumulate) {
    const size_t nmode = (size_t)c->M * c->M * c->Mh;
    {
        ScopedPhase ph(c, PSE_T_SPREAD);
        spread_kernel<<<c->ntile, 512, 0, c->stream>>>(c->d_pos, reinterpret_cast<const float4 *>(d_in), c->d_tile_start, c->d_tile_list,
                                                       c->d_grid, c->M, c->P, c->nt, (float)(1.0 / c->h), (float)(2.0 * M_PI / c->P));
        KERNEL_CHECK(c);
    }
    { ScopedPhase ph(c, PSE_T_FFT_FWD); CUFFT_TRY(c, cufftExecR2C(c->plan_r2c, c->d_grid, c->d_spec)); c->launches++; }
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        scale_kernel<<<(unsigned)((nmode + 255) / 256), 256, 0, c->stream>>>(c->d_spec, make_scale_params(c)); KERNEL_CHECK(c);
    }
    return inverse_and_interpolate(c, d_out, accumulate);
}

pse_status pse_wave_brownian(pse_ctx *c, const float *d_noise_wave, float *d_out, bool accumulate) {
    const size_t nmode = (size_t)c->M * c->M * c->Mh;
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        scale_brownian_kernel<<<(unsigned)((nmode + 255) / 256), 256, 0, c->stream>>>(
            c->d_spec, reinterpret_cast<const float2 *>(d_noise_wave), make_scale_params(c));
        KERNEL_CHECK(c);
    }
    return inverse_and_interpolate(c, d_out, accumulate);
}

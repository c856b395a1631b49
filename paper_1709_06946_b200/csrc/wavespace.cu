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
#include <algorithm>
#include <cuda_pipeline.h>
#include "pse_internal.h"
#include "wave_scale.cuh"

namespace {

constexpr int T = PSE_TILE;

__device__ __forceinline__ int support_base(float g, int P) { return pse_support_base(g, P); }
__device__ __forceinline__ int pmod(int i, int M) { return pse_pmod(i, M); }

// Exponent of the 1-D window at offset tt (grid units) from the particle.  wb == 0: the paper's Gaussian,
// exp(-wa tt^2) with wa = 2 pi / P.  wb > 0: "exponential of semicircle" window
// exp(wb (sqrt(1 - z^2) - 1)), z = 2 tt / P, wa = 4 / P^2 — same support, much faster decay in k, so a given
// tolerance needs fewer points per dimension.  The branch is uniform across the grid.
__device__ __forceinline__ float win_arg(float tt, float wa, float wb) {
    return wb > 0.f ? wb * (sqrtf(fmaxf(1.f - wa * tt * tt, 0.f)) - 1.f) : -wa * tt * tt;
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

constexpr int SPREAD_BATCH = 128, SPREAD_THREADS = 128;

// wrapped offset of grid point gp (0 <= gp < M) from an unwrapped support base (-P < base < M + P)
__device__ __forceinline__ int wrap_offset(int gp, int base, int M) {
    int o = gp - base;
    o += o < 0 ? M : 0;
    o -= o >= M ? M : 0;
    return o;
}

// 128 threads = 4 warps per 8^3 tile.  Warp w owns the x-planes 2w and 2w+1 (one per half-warp); inside a half-warp
// lane (b2 = bit 3, c = bits 0..2) owns the four points y = b2, b2+2, b2+4, b2+6 at z = c: 4 x 8 accumulators in
// registers, 32 FMAs per particle for ~18 other instructions.  Candidates are staged 128 at a time (one thread each:
// particle data + the 3 x 8 separable weights, y-weights stored permuted so that a lane's four are one float4), then
// compacted into one list per plane PAIR holding only the particles whose support covers it, in candidate order
// (fixed summation order, no atomics).
template <int C0, int NC>                           // components C0 .. C0+NC-1 are spread (0,8 | 0,3 | 3,5)
__global__ void __launch_bounds__(SPREAD_THREADS)
spread_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ in, const int *__restrict__ tile_start,
              const int *__restrict__ tile_list, float *__restrict__ grid, int M, int P, int nt, float inv_h, float wa, float wb) {
    __shared__ float4 q[SPREAD_BATCH][2];
    __shared__ __align__(16) float W[SPREAD_BATCH][3][T];
    __shared__ unsigned short lst[4][SPREAD_BATCH];
    __shared__ int cnt[4][5];                       // [plane pair][warp] counts -> exclusive prefix; [pair][4] = total
    __shared__ int bin_lo[64], bin_cum[65], nbins_s;
    __shared__ int reach[3][4], nreach[3];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int half = lane >> 4, b2 = (lane >> 3) & 1, cc = lane & 7, a = 2 * wid + half;
    const int t = blockIdx.x, t0 = t / (nt * nt), t1 = (t / nt) % nt, t2 = t % nt;
    const int g0[3] = {t0 * T, t1 * T, t2 * T};
    if (tid < 3) nreach[tid] = reach_tiles(tid == 0 ? t0 : (tid == 1 ? t1 : t2), M, P, nt, reach[tid]);
    __syncthreads();
    {
        const int ny = nreach[1], nz = nreach[2], n = nreach[0] * ny * nz;
        int cntb = 0;
        if (tid < n) {                                    // one thread per candidate bin: a single global round trip
            const int i = tid / (ny * nz), j = (tid / nz) % ny, k = tid % nz;
            const int tb = (reach[0][i] * nt + reach[1][j]) * nt + reach[2][k];
            const int lo = tile_start[tb];
            cntb = tile_start[tb + 1] - lo;
            bin_lo[tid] = lo;
        }
        int inc = cntb;                                   // n <= 64: inclusive scans in warps 0 and 1
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
        if (tid == 31) bin_cum[64] = inc;                 // total of warp 0, parked in the last slot
        if (tid < 32) bin_cum[tid] = inc - cntb;
        __syncthreads();
        if (wid == 1) { bin_cum[tid] = bin_cum[64] + inc - cntb; if (lane == 31) nbins_s = bin_cum[64] + inc; }
        __syncthreads();
        if (tid == 0) { const int tot = nbins_s; bin_cum[n] = tot; nbins_s = n; }
        __syncthreads();
    }
    const int nbins = nbins_s, total = bin_cum[nbins];
    float acc[4][NC];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[m][c] = 0.f;
    __shared__ int hs[2 * SPREAD_BATCH];            // particles whose support really reaches this tile, in candidate order
    __shared__ int hcnt[4];
    int nh = 0, cand = 0;                           // uniform over the CTA
    while (cand < total || nh > 0) {
        // phase 1: cheap geometric test on 128 candidates at a time (2 of 3 miss the tile), hits compacted into hs
        while (cand < total && nh <= SPREAD_BATCH) {
            const int ci = cand + tid;
            bool hit = false;
            int s = 0;
            if (ci < total) {
                int k = 0;
                while (bin_cum[k + 1] <= ci) ++k;
                s = tile_list[bin_lo[k] + ci - bin_cum[k]];
                const float4 p = pos[s];
                const float g[3] = {p.x * inv_h, p.y * inv_h, p.z * inv_h};
                hit = true;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const int o0 = wrap_offset(g0[d], support_base(g[d], P), M);
                    hit = hit && (o0 < P || o0 > M - T);
                }
            }
            const unsigned hb = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) hcnt[wid] = __popc(hb);
            __syncthreads();
            int woff = 0, tot = 0;
#pragma unroll
            for (int w = 0; w < 4; ++w) { const int v = hcnt[w]; woff += w < wid ? v : 0; tot += v; }
            if (hit) hs[nh + woff + __popc(hb & ((1u << lane) - 1))] = s;
            __syncthreads();
            nh += tot; cand += SPREAD_BATCH;
        }
        // phase 2: weights for up to 128 hits, one thread each (dense lanes)
        const int nb = min(nh, SPREAD_BATCH);
        unsigned xmask = 0;
        if (tid < nb) {
            const int s = hs[tid];
            const float4 p = pos[s];
            q[tid][0] = in[2 * s]; q[tid][1] = in[2 * s + 1];
            const float g[3] = {p.x * inv_h, p.y * inv_h, p.z * inv_h};
            unsigned msk[3] = {0u, 0u, 0u};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const int base = support_base(g[d], P);
#pragma unroll
                for (int i = 0; i < T; ++i) {
                    const int gp = g0[d] + i, o = wrap_offset(gp, base, M);
                    const float tt = (float)(base + o) - g[d];
                    const bool inside = (o < P && gp < M);
                    W[tid][d][d == 1 ? ((i & 1) * 4 + (i >> 1)) : i] = inside ? __expf(win_arg(tt, wa, wb)) : 0.f;
                    msk[d] |= inside ? (1u << i) : 0u;
                }
            }
            xmask = (msk[1] && msk[2]) ? msk[0] : 0u;
        }
        unsigned bal[4];
#pragma unroll
        for (int pr = 0; pr < 4; ++pr) bal[pr] = __ballot_sync(0xffffffffu, (xmask >> (2 * pr)) & 3u);
#pragma unroll
        for (int pr = 0; pr < 4; ++pr) if (lane == pr) cnt[pr][wid] = __popc(bal[pr]);
        __syncthreads();
        if (tid < 4) {                                            // exclusive prefix over the 4 warps, per plane pair
            int run = 0;
#pragma unroll
            for (int w = 0; w < 4; ++w) { const int v = cnt[tid][w]; cnt[tid][w] = run; run += v; }
            cnt[tid][4] = run;
        }
        __syncthreads();
        if (xmask) {
#pragma unroll
            for (int pr = 0; pr < 4; ++pr)
                if ((xmask >> (2 * pr)) & 3u) lst[pr][cnt[pr][wid] + __popc(bal[pr] & ((1u << lane) - 1))] = (unsigned short)tid;
        }
        __syncthreads();
        const int nact = cnt[wid][4];
        for (int i = 0; i < nact; ++i) {
            const int p = lst[wid][i];
            const float wxz = W[p][0][a] * W[p][2][cc];
            const float4 wy = *reinterpret_cast<const float4 *>(&W[p][1][4 * b2]);
            const float4 q0 = q[p][0], q1 = q[p][1];
            const float w[4] = {wxz * wy.x, wxz * wy.y, wxz * wy.z, wxz * wy.w};
            const float qv[8] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
#pragma unroll
            for (int m = 0; m < 4; ++m)
#pragma unroll
                for (int c = 0; c < NC; ++c) acc[m][c] += w[m] * qv[C0 + c];
        }
        __syncthreads();
        const int left = nh - nb;                     // leftover hits (<= 128) move to the front of the buffer
        const int mv = tid < left ? hs[nb + tid] : 0;
        __syncthreads();
        if (tid < left) hs[tid] = mv;
        __syncthreads();
        nh = left;
    }
    const int gx = g0[0] + a, gz = g0[2] + cc;
    const size_t M3 = pse_plane_stride(M);
    if (gx < M && gz < M) {
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const int gy = g0[1] + b2 + 2 * m;
            if (gy < M) {
                const size_t o = ((size_t)gx * M + gy) * M + gz;
#pragma unroll
                for (int c = 0; c < NC; ++c) grid[(C0 + c) * M3 + o] = acc[m][c];
            }
        }
    }
}

// Interpolation (a7): warp per particle (visited in tile order for L1/L2 locality), lanes over the P^3 support.
__global__ void __launch_bounds__(256)
interp_kernel(const float4 *__restrict__ pos, const int *__restrict__ tile_list, const float *__restrict__ grid,
              float4 *__restrict__ out, int N, int M, int P, float inv_h, float wa, float wb, int accumulate, int mode) {
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
        wr[h] = (d < 3) ? __expf(win_arg(tt, wa, wb)) : 0.f;
    }
    const size_t M3 = pse_plane_stride(M);
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
            for (int c = 0; c < 8; ++c)
                if (mode & (c < 3 ? PSE_OUT_U : PSE_OUT_E)) acc[c] += w * __ldg(grid + c * M3 + o);
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

// Interpolation, tile-staged (default path): one CTA per tile bin.  The (T+P-1)^3 block of all 8 grids that the
// bin's particles can touch is staged once in shared memory with coalesced loads (periodic wrap resolved while
// loading), then each warp takes particles of the bin, lanes over the P^3 support, reading only shared memory.
// Every particle belongs to exactly one bin, so the output is written once, with no atomics.
template <int PT>                                  // PT > 0: support size known at compile time (no integer divisions)
__global__ void __launch_bounds__(256)
interp_tile_kernel(const float4 *__restrict__ pos, const int *__restrict__ tile_start, const int *__restrict__ tile_list,
                   const float *__restrict__ grid, float4 *__restrict__ out, int M, int Prt, int nt, float inv_h, float wa, float wb,
                   int accumulate, int mode) {
    extern __shared__ float4 sm[];
    const int P = PT ? PT : Prt;
    const int E = T + P - 1, Ez = E + ((P - E) & 7), E3 = E * E * Ez;   // z-rows padded so that Ez = P (mod 8): the
    float4 *lo = sm, *hi = sm + E3;                                      // 16-byte chunks of a (j,k) lane set never collide
    const int t = blockIdx.x, t0 = t / (nt * nt), t1 = (t / nt) % nt, t2 = t % nt;
    const int first = tile_start[t], np = tile_start[t + 1] - first;
    if (np == 0) return;
    const size_t M3 = pse_plane_stride(M);
    {   // stage row by row: a half-warp (E <= 16) or a warp per (ix,iy) row, lanes along z; wrap by subtraction
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
        const int rpi = E <= 16 ? 2 : 1, lz = E <= 16 ? (lane & 15) : lane, sub = E <= 16 ? (lane >> 4) : 0;
        int gz = t2 * T + lz;
        while (gz >= M) gz -= M;
        for (int row = wid * rpi + sub; row < E * E; row += nw * rpi) {
            const int ix = row / E, iy = row - ix * E;
            int gx = t0 * T + ix, gy = t1 * T + iy;
            while (gx >= M) gx -= M;
            while (gy >= M) gy -= M;
            if (lz < E) {
                const size_t o = ((size_t)gx * M + gy) * M + gz;
                const int idx = row * Ez + lz;
                // asynchronous 4-byte copies global -> shared (cp.async, LDGSTS): all rows of the block are in flight
                // at once instead of one L2 round trip per row; planes the caller did not ask for are zero-filled
                float *dlo = reinterpret_cast<float *>(lo + idx), *dhi = reinterpret_cast<float *>(hi + idx);
                if (mode & PSE_OUT_U) {
                    __pipeline_memcpy_async(dlo, grid + o, 4); __pipeline_memcpy_async(dlo + 1, grid + M3 + o, 4);
                    __pipeline_memcpy_async(dlo + 2, grid + 2 * M3 + o, 4);
                } else { dlo[0] = 0.f; dlo[1] = 0.f; dlo[2] = 0.f; }
                if (mode & PSE_OUT_E) {
                    __pipeline_memcpy_async(dlo + 3, grid + 3 * M3 + o, 4);
                    __pipeline_memcpy_async(dhi, grid + 4 * M3 + o, 4); __pipeline_memcpy_async(dhi + 1, grid + 5 * M3 + o, 4);
                    __pipeline_memcpy_async(dhi + 2, grid + 6 * M3 + o, 4); __pipeline_memcpy_async(dhi + 3, grid + 7 * M3 + o, 4);
                } else { dlo[3] = 0.f; hi[idx] = make_float4(0.f, 0.f, 0.f, 0.f); }
            }
        }
        __pipeline_commit();
        __pipeline_wait_prior(0);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int P2 = P * P, EE = E * Ez;
    float *outf = reinterpret_cast<float *>(out);
    // Eight lanes per particle, four particles per warp.  A lane owns the (j,k) columns jk = gl, gl + 8, ... of the
    // support and walks each along x: two 16-byte shared loads and 8 FMAs per point, the x weights in registers.  The
    // fixed cost per particle (support base, weights, reduction, read-modify-write) is paid by 8 lanes instead of 32,
    // and the 8-lane reduction leaves component gl in lane gl: one 32-byte store per particle.
    constexpr int NP = PT ? PT : PSE_MAXP;
    const int gl = lane & 7, grp = lane >> 3, gbase = lane & 24;
    const bool mine = mode & (gl < 3 ? PSE_OUT_U : PSE_OUT_E);
    for (int pi0 = wid * 4; pi0 < np; pi0 += nw * 4) {                  // uniform over the warp (shuffles inside)
        const int pi = pi0 + grp;
        const bool live = pi < np;
        const int s = live ? tile_list[first + pi] : 0;
        const float4 p = pos[s];
        const float prev = (live && mine && accumulate) ? outf[(size_t)s * 8 + gl] : 0.f;       // read-modify-write operand early
        const float gx = p.x * inv_h, gy = p.y * inv_h, gz = p.z * inv_h;
        const int b0 = support_base(gx, P), b1 = support_base(gy, P), b2 = support_base(gz, P);
        const int r0 = pmod(b0, M) - t0 * T, r1 = pmod(b1, M) - t1 * T, r2 = pmod(b2, M) - t2 * T;
        // x weights: lane gl evaluates i = gl (and gl + 8 for supports wider than 8), the group shares them by shuffle
        const float wxa = gl < P ? __expf(win_arg((float)(b0 + gl) - gx, wa, wb)) : 0.f;
        const float wxb = (NP > 8 && gl + 8 < P) ? __expf(win_arg((float)(b0 + gl + 8) - gx, wa, wb)) : 0.f;
        float wx[NP];
#pragma unroll
        for (int i = 0; i < NP; ++i) wx[i] = __shfl_sync(0xffffffffu, i < 8 ? wxa : wxb, gbase + (i & 7));
        float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const int ncol = live ? P2 : 0;
        for (int jk = gl; jk < ncol; jk += 8) {
            const int j = jk / P, k = jk - j * P;
            const float wyz = __expf(win_arg((float)(b1 + j) - gy, wa, wb) + win_arg((float)(b2 + k) - gz, wa, wb));
            int sidx = (r0 * E + r1 + j) * Ez + r2 + k;
            float tsum[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
            for (int i = 0; i < NP; ++i) {
                if (i >= P) break;
                const float4 v0 = lo[sidx], v1 = hi[sidx];
                tsum[0] += wx[i] * v0.x; tsum[1] += wx[i] * v0.y; tsum[2] += wx[i] * v0.z; tsum[3] += wx[i] * v0.w;
                tsum[4] += wx[i] * v1.x; tsum[5] += wx[i] * v1.y; tsum[6] += wx[i] * v1.z; tsum[7] += wx[i] * v1.w;
                sidx += EE;
            }
#pragma unroll
            for (int c = 0; c < 8; ++c) acc[c] += wyz * tsum[c];
        }
        // 8 sums over 8 lanes in 4 + 2 + 1 shuffles: every step halves the values a lane carries
        const bool h4 = gl & 4, h2 = gl & 2, h1 = gl & 1;
        float r4[4], r2s[2];
#pragma unroll
        for (int c = 0; c < 4; ++c) r4[c] = (h4 ? acc[c + 4] : acc[c]) + __shfl_xor_sync(0xffffffffu, h4 ? acc[c] : acc[c + 4], 4);
#pragma unroll
        for (int c = 0; c < 2; ++c) r2s[c] = (h2 ? r4[c + 2] : r4[c]) + __shfl_xor_sync(0xffffffffu, h2 ? r4[c] : r4[c + 2], 2);
        const float r = (h1 ? r2s[1] : r2s[0]) + __shfl_xor_sync(0xffffffffu, h1 ? r2s[0] : r2s[1], 1);
        if (live && mine) outf[(size_t)s * 8 + gl] = r + prev;
    }
}

// a5 (cuFFT path): one thread per half-spectrum mode, in place
// (grid.y = ix, grid.x covers the (iy, iz) plane: 32-bit index arithmetic, no 64-bit division per thread)
__global__ void __launch_bounds__(256) scale_kernel(cufftComplex *spec, ScaleParams sp) {
    const unsigned plane = (unsigned)sp.M * (unsigned)sp.Mh, rem = blockIdx.x * blockDim.x + threadIdx.x;
    if (rem >= plane) return;
    const int ix = (int)blockIdx.y, iy = (int)(rem / (unsigned)sp.Mh), iz = (int)(rem - (unsigned)iy * (unsigned)sp.Mh);
    const size_t nmode = (size_t)plane * sp.M, o = (size_t)ix * plane + rem;
    scale_point(sp, ix, iy, iz, spec, nmode, o, spec, nmode, o);
}

// a5, Brownian flavour (Eq. 75): uh = c_br sqrt((1+k^2/4xi^2)/(eta k^2)) exp(-(1-eta_g) k^2/8xi^2) (I - kh kh) W(k),
// W(k) = (g_re + i g_im)/sqrt2 from the noise buffer; in the plane kz = 0 the non-canonical member of each +-k
// pair takes the conjugate of its partner's entry (reading R8) so that the C2R transform sees a Hermitian field.
__global__ void __launch_bounds__(256) scale_brownian_kernel(cufftComplex *spec, const float2 *__restrict__ noise, ScaleParams sp) {
    const int M = sp.M;
    const unsigned plane = (unsigned)M * (unsigned)sp.Mh, rem = blockIdx.x * blockDim.x + threadIdx.x;
    if (rem >= plane) return;
    const int ix = (int)blockIdx.y, iy = (int)(rem / (unsigned)sp.Mh), iz = (int)(rem - (unsigned)iy * (unsigned)sp.Mh);
    const size_t nmode = (size_t)plane * M, o = (size_t)ix * plane + rem;
    float kx, ky, kz;
    float2 zero = make_float2(0.f, 0.f);
    const size_t oplane = nmode, oo = o;
    if (!mode_k(sp, ix, iy, iz, kx, ky, kz)) {
#pragma unroll
        for (int c = 0; c < 8; ++c) spec[c * oplane + oo] = zero;
        return;
    }
    const int half = (M + 1) / 2, nx = ix < half ? ix : ix - M, ny = iy < half ? iy : iy - M;
    const bool canon = iz > 0 || ny > 0 || (ny == 0 && nx > 0);
    const size_t src = canon ? o : ((size_t)((M - ix) % M) * M + (size_t)((M - iy) % M)) * sp.Mh;
    const float sgn = canon ? 1.f : -1.f;
    float2 W[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { float2 g = noise[c * nmode + src]; W[c] = make_float2(g.x * WS_RS2, sgn * g.y * WS_RS2); }
    const float k2 = kx * kx + ky * ky + kz * kz, kn = sqrtf(k2), ka = kn * sp.a;
    float s0, s1;
    shape_factors(ka, s0, s1);
    const float q = k2 * sp.inv4xi2;
    const float Bh = sp.c_br * sqrtf(sp.inv_eta * (1.f + q) / k2) * __expf(-0.5f * q) * __ldg(sp.dec + ix) * __ldg(sp.dec + iy) * __ldg(sp.dec + iz);
    const float ik2 = 1.f / k2;
    const float2 kw = make_float2((kx * W[0].x + ky * W[1].x + kz * W[2].x) * ik2, (kx * W[0].y + ky * W[1].y + kz * W[2].y) * ik2);
    const float2 ux = make_float2(Bh * (W[0].x - kx * kw.x), Bh * (W[0].y - kx * kw.y));
    const float2 uy = make_float2(Bh * (W[1].x - ky * kw.x), Bh * (W[1].y - ky * kw.y));
    const float2 uz = make_float2(Bh * (W[2].x - kz * kw.x), Bh * (W[2].y - kz * kw.y));
    write_outputs(spec, oplane, oo, s0, s1, kx, ky, kz, ux, uy, uz, PSE_OUT_U | PSE_OUT_E);
}

}  // namespace

pse_status pse_wave_init(pse_ctx *c) {
    const int M = c->M;
    c->Mh = M / 2 + 1;
    c->nt = (M + T - 1) / T; c->ntile = c->nt * c->nt * c->nt;
    const size_t M3 = pse_plane_stride(M), nmode = (size_t)M * M * c->Mh;
    CUDA_TRY(c, cudaMalloc(&c->d_grid, 8 * M3 * sizeof(float)));
    CUDA_TRY(c, cudaMalloc(&c->d_spec, 8 * nmode * sizeof(cufftComplex)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_start, (size_t)(c->ntile + 1) * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_of, (size_t)c->N * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_list, (size_t)c->N * sizeof(int)));
    int n[3] = {M, M, M};
    const int batches[3] = {8, 3, 5};                 // all grids | planes 0-2 (F in, U out) | planes 3-7 (S in, E out)
    size_t w = 0;
    for (int i = 0; i < 3; ++i) {
        size_t w1 = 0, w2 = 0;
        CUFFT_TRY(c, cufftCreate(&c->plan_r2c[i])); CUFFT_TRY(c, cufftCreate(&c->plan_c2r[i])); c->nplans = i + 1;
        CUFFT_TRY(c, cufftSetAutoAllocation(c->plan_r2c[i], 0)); CUFFT_TRY(c, cufftSetAutoAllocation(c->plan_c2r[i], 0));
        if (M3 == (size_t)M * M * M) {                // even M: packed planes, basic layout
            CUFFT_TRY(c, cufftMakePlanMany(c->plan_r2c[i], 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, batches[i], &w1));
            CUFFT_TRY(c, cufftMakePlanMany(c->plan_c2r[i], 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, batches[i], &w2));
        } else {                                      // odd M: real planes pse_plane_stride(M) apart
            int nr[3] = {M, M, M}, ncx[3] = {M, M, c->Mh};
            CUFFT_TRY(c, cufftMakePlanMany(c->plan_r2c[i], 3, n, nr, 1, (int)M3, ncx, 1, M * M * c->Mh, CUFFT_R2C, batches[i], &w1));
            CUFFT_TRY(c, cufftMakePlanMany(c->plan_c2r[i], 3, n, ncx, 1, M * M * c->Mh, nr, 1, (int)M3, CUFFT_C2R, batches[i], &w2));
        }
        w = std::max(w, std::max(w1, w2));
    }
    if (w) CUDA_TRY(c, cudaMalloc(&c->d_fft_work, w));
    for (int i = 0; i < 3; ++i) {
        CUFFT_TRY(c, cufftSetWorkArea(c->plan_r2c[i], c->d_fft_work)); CUFFT_TRY(c, cufftSetWorkArea(c->plan_c2r[i], c->d_fft_work));
        CUFFT_TRY(c, cufftSetStream(c->plan_r2c[i], c->stream)); CUFFT_TRY(c, cufftSetStream(c->plan_c2r[i], c->stream));
    }
    return PSE_OK;
}

void pse_wave_free(pse_ctx *c) {
    for (int i = 0; i < c->nplans; ++i) { cufftDestroy(c->plan_r2c[i]); cufftDestroy(c->plan_c2r[i]); }
    cudaFree(c->d_grid); cudaFree(c->d_spec); cudaFree(c->d_fft_work);
    cudaFree(c->d_tile_start); cudaFree(c->d_tile_of); cudaFree(c->d_tile_list);
}

// Tile bins: counted in wrap_and_bin, scanned with the cell counts, scattered in gather_positions (neighbors.cu);
// what is left is the deterministic order inside every tile.
pse_status pse_tile_bins(pse_ctx *c) {
    return pse_rank_sort(c, c->d_tile_start, c->ntile, c->d_tile_tmp, c->d_tile_list);
}

// plane range of a 2-bit component mask (bit 0: planes 0-2, bit 1: planes 3-7): plan index and first plane
static inline void plane_range(int bits, int &plan, int &first) {
    plan = bits == 3 ? 0 : bits; first = bits == 2 ? 3 : 0;
}

static pse_status inverse_and_interpolate(pse_ctx *c, float *d_out, bool accumulate, int mode = PSE_MODE_ALL) {
    {
        ScopedPhase ph(c, PSE_T_FFT_INV);
        int plan, first;
        plane_range((mode >> 2) & 3, plan, first);
        const size_t M3 = pse_plane_stride(c->M), nmode = (size_t)c->M * c->M * c->Mh;
        CUFFT_TRY(c, cufftExecC2R(c->plan_c2r[plan], c->d_spec + first * nmode, c->d_grid + first * M3)); c->launches++;
    }
    ScopedPhase ph(c, PSE_T_INTERP);
    const int TB = 256, E = T + c->P - 1;
    const int Ez = E + ((c->P - E) & 7);
    const size_t smem = (size_t)2 * E * E * Ez * sizeof(float4);
    if (smem <= 200 * 1024) {
#define PSE_LAUNCH_INTERP(PT)                                                                                              \
    do {                                                                                                                   \
        static size_t smem_set = 0;                                                                                        \
        if (smem > smem_set) {                                                                                             \
            CUDA_TRY(c, cudaFuncSetAttribute(interp_tile_kernel<PT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
            smem_set = smem;                                                                                               \
        }                                                                                                                  \
        interp_tile_kernel<PT><<<c->ntile, TB, smem, c->stream>>>(c->d_pos, c->d_tile_start, c->d_tile_list, c->d_grid,       \
            reinterpret_cast<float4 *>(d_out), c->M, c->P, c->nt, (float)(1.0 / c->h), (float)c->win_a, (float)c->win_b, \
            accumulate ? 1 : 0, mode);                                                                                     \
    } while (0)
        switch (c->P) {
            case 3: PSE_LAUNCH_INTERP(3); break;
            case 4: PSE_LAUNCH_INTERP(4); break;
            case 5: PSE_LAUNCH_INTERP(5); break;
            case 6: PSE_LAUNCH_INTERP(6); break;
            case 7: PSE_LAUNCH_INTERP(7); break;
            case 8: PSE_LAUNCH_INTERP(8); break;
            default: PSE_LAUNCH_INTERP(0); break;
        }
#undef PSE_LAUNCH_INTERP
    } else {
        interp_kernel<<<(unsigned)(((size_t)c->N * 32 + TB - 1) / TB), TB, 0, c->stream>>>(
            c->d_pos, c->d_tile_list, c->d_grid, reinterpret_cast<float4 *>(d_out), c->N, c->M, c->P, (float)(1.0 / c->h),
            (float)c->win_a, (float)c->win_b, accumulate ? 1 : 0, mode);
    }
    KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_wave_apply(pse_ctx *c, const float *d_in, float *d_out, bool accumulate, int mode) {
    const size_t nmode = (size_t)c->M * c->M * c->Mh, M3 = pse_plane_stride(c->M);
    if (!(mode & (PSE_IN_F | PSE_IN_S)) || !(mode & (PSE_OUT_U | PSE_OUT_E))) { c->err = "pse_wave_apply: empty component mask"; return PSE_EINVAL; }
    int plan, first;
    plane_range(mode & 3, plan, first);
    {
        ScopedPhase ph(c, PSE_T_SPREAD);
        const float4 *in4 = reinterpret_cast<const float4 *>(d_in);
        const float ih = (float)(1.0 / c->h), wa = (float)c->win_a, wb = (float)c->win_b;
        if (plan == 0) spread_kernel<0, 8><<<c->ntile, SPREAD_THREADS, 0, c->stream>>>(c->d_pos, in4, c->d_tile_start, c->d_tile_list, c->d_grid, c->M, c->P, c->nt, ih, wa, wb);
        else if (plan == 1) spread_kernel<0, 3><<<c->ntile, SPREAD_THREADS, 0, c->stream>>>(c->d_pos, in4, c->d_tile_start, c->d_tile_list, c->d_grid, c->M, c->P, c->nt, ih, wa, wb);
        else spread_kernel<3, 5><<<c->ntile, SPREAD_THREADS, 0, c->stream>>>(c->d_pos, in4, c->d_tile_start, c->d_tile_list, c->d_grid, c->M, c->P, c->nt, ih, wa, wb);
        KERNEL_CHECK(c);
    }
    { ScopedPhase ph(c, PSE_T_FFT_FWD); CUFFT_TRY(c, cufftExecR2C(c->plan_r2c[plan], c->d_grid + first * M3, c->d_spec + first * nmode)); c->launches++; }
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        scale_kernel<<<dim3((unsigned)((c->M * c->Mh + 255) / 256), (unsigned)c->M), 256, 0, c->stream>>>(c->d_spec, make_scale_params(c, mode)); KERNEL_CHECK(c);
    }
    return inverse_and_interpolate(c, d_out, accumulate, mode);
}

pse_status pse_wave_brownian(pse_ctx *c, const float *d_noise_wave, float *d_out, bool accumulate) {
    const size_t nmode = (size_t)c->M * c->M * c->Mh;
    if (c->noise_pending) { CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->ev_noise, 0)); c->noise_pending = false; }
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        scale_brownian_kernel<<<dim3((unsigned)((c->M * c->Mh + 255) / 256), (unsigned)c->M), 256, 0, c->stream>>>(
            c->d_spec, reinterpret_cast<const float2 *>(d_noise_wave), make_scale_params(c));
        KERNEL_CHECK(c);
    }
    return inverse_and_interpolate(c, d_out, accumulate);
}

// Wave-space half of the product: M_w = sigma Q^T F^H P^H B P F Q (Eq. 42) and the Brownian factor
// M_w^{1/2} = sigma^{1/2} Q^T F^H P^H B^{1/2} (Eq. 75).  Steps a3-a7 of SURVEY.md §8(a).
//
// Grid layout: 8 planar real grids [c][ix][iy][iz] (iz fastest, planes pse_plane_stride(M) floats apart), grid point n at
// n*h; half spectrum [c][ix][iy][iz<=M/2].  c = (Fx,Fy,Fz,S1..S5) going in, (Ux,Uy,Uz,E1..E5) coming out.
// Window of Q / Q^T on its P^3 support (R3-R5): exponential of semicircle by default, the paper's Gaussian
// exp(-(2 pi/P) t^2) (eta_g = (h P xi/m)^2, m = sqrt(pi P)) on request; its continuous transform is divided out
// per dimension in the scale kernels (table d_dec), together with 1/V, so all normalisation lives there.
//
// What runs where:
//   pse_neighbors   particle_window_kernel (support base + window values per particle, tile order), half_lists_kernel
//   spread          spread_blocks_kernel (P <= 8: lane owns 2x2x2 grid points, gather form, register accumulators, lists),
//                   spread_kernel (generic gather for wider supports / tiny grids); no atomics, no memset, fixed order
//   scale           scale_kernel (P^H B P), scale_brownian_kernel (P^H B^{1/2} W on the finer grid of the Brownian pass)
//   interpolate     interp_planes_kernel (P <= 8: TMA-staged tile block, 8 lanes per particle), interp_kernel (generic)
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

// ---- per-particle window data -------------------------------------------------------------------------------------------
// Positions are fixed between two pse_neighbors calls while ~25 spreads / interpolations run on them, so the P window values
// per dimension (a sqrt and an exp each for the default window) and the wrapped support base are computed once here.  Both
// arrays are in TILE ORDER (entry i belongs to particle tile_list[i]): the particles of a tile bin are contiguous, so spread
// and interpolation read them without an indirection.
template <int PP>
__global__ void particle_window_kernel(const float4 *__restrict__ pos, const int *__restrict__ tile_list, int N, int M, int P, float inv_h,
                                       float wa, float wb, int *__restrict__ pbase, float4 *__restrict__ pw) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 p = pos[tile_list[i]];
    const float g[3] = {p.x * inv_h, p.y * inv_h, p.z * inv_h};
    int packed = 0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int base = support_base(g[d], P);
        packed |= pmod(base, M) << (10 * d);
        float v[PP];
#pragma unroll
        for (int k = 0; k < PP; ++k) v[k] = k < P ? __expf(win_arg((float)(base + k) - g[d], wa, wb)) : 0.f;
#pragma unroll
        for (int k4 = 0; k4 < PP / 4; ++k4) pw[((size_t)i * 3 + d) * (PP / 4) + k4] = make_float4(v[4 * k4], v[4 * k4 + 1], v[4 * k4 + 2], v[4 * k4 + 3]);
    }
    pbase[i] = packed;
}

// ---- tile bins of the finer grid of the Brownian pass (built on demand, once per configuration that draws a sample) ----
__global__ void fine_bin_count(const float4 *__restrict__ pos, int N, float inv_h, int M, int P, int nt, int *__restrict__ tile_of, int *__restrict__ count) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const int t = pse_tile_of(pos[s], inv_h, M, P, nt);
    tile_of[s] = t;
    atomicAdd(count + t, 1);
}
__global__ void fine_bin_scatter(const int *__restrict__ tile_of, int N, const int *__restrict__ start, int *__restrict__ fill, int *__restrict__ tmp) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const int t = tile_of[s];
    tmp[start[t] + atomicAdd(fill + t, 1)] = s;                      // order inside a tile fixed afterwards by the rank sort
}

// ---- lists of the particles that reach each half tile (built once per pse_neighbors, used by every spread) -----------------
// A "half" is the 4 x 8 x 8 block of grid points one warp of the spread kernel owns: half index = (tile index) * 2 + (x half).
// One warp per half walks the tile bins that can reach it (two per dimension, three next to a partial last tile), 32 entries
// at a time, keeps the particles whose support overlaps the half and collects them in bin order with a ballot (no atomics per
// particle, deterministic content).  The warp then reserves its segment of the list array with ONE atomicAdd on a cursor (the
// placement of whole segments depends on scheduling, which no consumer sees: they go through half_start / half_count) and
// copies the collected entries out.  Entries are tile-order indices (see particle_window_kernel).
constexpr int HL_WARPS = 4, HL_CAP = 512;

__global__ void __launch_bounds__(HL_WARPS * 32)
half_lists_kernel(const int *__restrict__ pbase, const int *__restrict__ tile_start, int M, int P, int nt, int nhalf,
                  int *__restrict__ half_start, int *__restrict__ half_count, int *__restrict__ half_list, int *__restrict__ cursor) {
    __shared__ int s_hits[HL_WARPS][HL_CAP];
    __shared__ int s_reach[HL_WARPS][3][4], s_nreach[HL_WARPS][3];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, h = blockIdx.x * HL_WARPS + w;
    if (h >= nhalf) return;
    const int t = h >> 1, t0 = t / (nt * nt), t1 = (t / nt) % nt, t2 = t % nt;
    const int lo[3] = {t0 * T + 4 * (h & 1), t1 * T, t2 * T};
    if (lane < 3) s_nreach[w][lane] = reach_tiles(lane == 0 ? t0 : (lane == 1 ? t1 : t2), M, P, nt, s_reach[w][lane]);
    __syncwarp();
    const int nx = s_nreach[w][0], ny = s_nreach[w][1], nz = s_nreach[w][2];
    const int halfM = M >> 1;
    int found = 0, base_out = 0;
    // pass 0 collects in shared memory (and counts); only if the half holds more than HL_CAP particles a second pass writes the rest
    for (int pass = 0; pass < 2; ++pass) {
        int seen = 0;
        for (int bi = 0; bi < nx * ny * nz; ++bi) {
            const int i = bi / (ny * nz), j = (bi / nz) % ny, k = bi % nz;
            const int tb = (s_reach[w][0][i] * nt + s_reach[w][1][j]) * nt + s_reach[w][2][k];
            const int first = tile_start[tb], cnt = tile_start[tb + 1] - first;
            for (int c0 = 0; c0 < cnt; c0 += 32) {
                const int e = first + c0 + lane;
                bool hit = c0 + lane < cnt;
                if (hit) {
                    const int b = pbase[e];
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        int so = lo[d] - ((b >> (10 * d)) & 1023);                  // offset of the half's origin from the support base
                        so += so < -halfM ? M : 0;
                        so -= so > halfM ? M : 0;
                        hit = hit && so > -(d == 0 ? 4 : 8) && so < P;
                    }
                }
                const unsigned bal = __ballot_sync(0xffffffffu, hit);
                const int at = seen + __popc(bal & ((1u << lane) - 1u));
                if (hit) {
                    if (pass == 0) { if (at < HL_CAP) s_hits[w][at] = e; }
                    else if (at >= HL_CAP) half_list[base_out + at] = e;
                }
                seen += __popc(bal);
            }
        }
        if (pass == 0) {
            found = seen;
            if (lane == 0) { base_out = atomicAdd(cursor, found); half_start[h] = base_out; half_count[h] = found; }
            base_out = __shfl_sync(0xffffffffu, base_out, 0);
            __syncwarp();
            for (int q = lane; q < min(found, HL_CAP); q += 32) half_list[base_out + q] = s_hits[w][q];
            if (found <= HL_CAP) break;
        }
    }
}

// ---- spread (a3), default path for P <= 8 ---------------------------------------------------------------------------------
// Gather form with REGISTER accumulators, as before, but with the lane footprint matched to the support: a lane owns a
// 2 x 2 x 2 block of grid points (8 points x NC components in registers), a warp a 4 x 8 x 8 half of an 8^3 tile, and a lane
// evaluates a particle only if the particle's P^3 support really overlaps its block: (P/(P+1))^3 = 51 % of its FMAs are then
// useful at P = 4, against 17 % when a half-warp owned a whole 8 x 8 face (ncu, round 1).  Per warp, with no CTA barrier:
//   1. the particles that reach the warp's half come from the list built in pse_neighbors, 32 at a time, one per lane: the
//      lane stages its particle in shared memory (inputs, zero-padded window rows, the offset of the half's origin from the
//      support base, and a 10-bit code of the blocks the support overlaps per dimension);
//   2. every lane builds a 64-bit mask of the staged particles whose code covers its own block (one AND + compare each);
//   3. every lane walks its own mask: 6 window values, 12 products, 8 x NC FMAs per entry.
// No atomics, no memset, each grid value written once (8-byte stores), summation in list order (deterministic).
template <int P, int C0, int NC>
__global__ void __launch_bounds__(64)
spread_blocks_kernel(const int *__restrict__ pbase, const float *__restrict__ pw, const int *__restrict__ tile_list, const float4 *__restrict__ in,
                     const int *__restrict__ half_start, const int *__restrict__ half_count, const int *__restrict__ half_list,
                     float *__restrict__ grid, int M, int nt) {
    constexpr int CAP = 64, PP = (P + 3) & ~3, WR = P + 2, WROW = (3 * WR) | 1, QROW = 3;     // odd row pitch (words) / 48-byte rows:
    __shared__ __align__(16) unsigned s_code[2][CAP];                                         // lanes on different rows, different banks
    __shared__ unsigned s_off[2][CAP];
    __shared__ float4 s_q[2][CAP][QROW];
    __shared__ float s_w[2][CAP][WROW];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int t = blockIdx.x, t0 = t / (nt * nt), t1 = (t / nt) % nt, t2 = t % nt;
    const int lo[3] = {t0 * T + 4 * w, t1 * T, t2 * T};            // origin of the warp's half: 4 x 8 x 8 points
    const int first = half_start[2 * t + w], total = half_count[2 * t + w];
    const int rxl = lane >> 4, ryl = (lane >> 2) & 3, rzl = lane & 3;            // my block inside the half: 2 x 4 x 4 blocks
    const unsigned mymask = (1u << rxl) | (1u << (2 + ryl)) | (1u << (6 + rzl));
    const int cx = 2 * rxl + 1 - 16, cy = 2 * ryl + 1 - 16, cz = 2 * rzl + 1 - 16;
    const int halfM = M >> 1;
    float acc[8][NC];
#pragma unroll
    for (int m = 0; m < 8; ++m)
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[m][c] = 0.f;
    for (int c0 = 0; c0 < total; c0 += CAP) {
        const int nb = min(CAP, total - c0);
        // 1. stage up to CAP particles of the list, one per lane and pass
#pragma unroll
        for (int pass = 0; pass < CAP / 32; ++pass) {
            const int slot = pass * 32 + lane;
            if (slot < nb) {
                const int e = half_list[first + c0 + slot];          // tile-order index: window data contiguous per tile
                const int b = pbase[e], s = tile_list[e];
                unsigned code = 0, off = 0;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const int nblk = d == 0 ? 2 : 4, sh = d == 0 ? 0 : (d == 1 ? 2 : 6);
                    int so = lo[d] - ((b >> (10 * d)) & 1023);                  // offset of the half's origin from the support base,
                    so += so < -halfM ? M : 0;                                  // minimum image: -len < so < P for a listed particle
                    so -= so > halfM ? M : 0;
                    const int rmin = max(0, (-so) >> 1), rmax = min(nblk - 1, (P - 1 - so) >> 1);      // blocks r with -1-2r <= so <= P-1-2r
                    code |= (((2u << rmax) - 1u) & ~((1u << rmin) - 1u)) << sh;
                    off |= (unsigned)((so + 16) & 255) << (8 * d);
                }
                s_code[w][slot] = code; s_off[w][slot] = off;
                s_q[w][slot][0] = in[2 * s]; s_q[w][slot][1] = in[2 * s + 1];
                const float4 *src = reinterpret_cast<const float4 *>(pw + (size_t)e * 3 * PP);
                float *dst = s_w[w][slot];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    float v[PP];
#pragma unroll
                    for (int i4 = 0; i4 < PP / 4; ++i4) { const float4 x = src[d * (PP / 4) + i4]; v[4 * i4] = x.x; v[4 * i4 + 1] = x.y; v[4 * i4 + 2] = x.z; v[4 * i4 + 3] = x.w; }
                    dst[d * WR] = 0.f;
#pragma unroll
                    for (int i = 0; i < P; ++i) dst[d * WR + 1 + i] = v[i];
                    dst[d * WR + P + 1] = 0.f;
                }
            } else if (slot < ((nb + 3) & ~3)) s_code[w][slot] = 0u;            // padding of the last group of four codes
        }
        __syncwarp();
        // 2. my particles of this batch as a bit mask (four codes per 16-byte shared load)
        unsigned mlo = 0u, mhi = 0u;
#pragma unroll
        for (int i4 = 0; i4 < CAP / 4; ++i4) {
            if (4 * i4 < nb) {
                const uint4 cd = *reinterpret_cast<const uint4 *>(&s_code[w][4 * i4]);
                const unsigned bits = ((cd.x & mymask) == mymask ? 1u : 0u) | ((cd.y & mymask) == mymask ? 2u : 0u) |
                                      ((cd.z & mymask) == mymask ? 4u : 0u) | ((cd.w & mymask) == mymask ? 8u : 0u);
                if (i4 < 8) mlo |= bits << (4 * i4); else mhi |= bits << (4 * (i4 - 8));
            }
        }
        unsigned long long m = ((unsigned long long)mhi << 32) | mlo;
        // 3. walk the mask
        while (m) {
            const int i = __ffsll((long long)m) - 1;
            m &= m - 1ull;
            const unsigned off = s_off[w][i];
            const float *wr = s_w[w][i];
            const int ix = (int)(off & 255u) + cx, iy = (int)((off >> 8) & 255u) + cy, iz = (int)((off >> 16) & 255u) + cz;
            const float wx0 = wr[ix], wx1 = wr[ix + 1], wy0 = wr[WR + iy], wy1 = wr[WR + iy + 1], wz0 = wr[2 * WR + iz], wz1 = wr[2 * WR + iz + 1];
            const float4 q0 = s_q[w][i][0], q1 = s_q[w][i][1];
            const float qv[8] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
            const float wxy[4] = {wx0 * wy0, wx0 * wy1, wx1 * wy0, wx1 * wy1};
#pragma unroll
            for (int ab = 0; ab < 4; ++ab) {
                const float w0 = wxy[ab] * wz0, w1 = wxy[ab] * wz1;
#pragma unroll
                for (int c = 0; c < NC; ++c) { acc[2 * ab][c] += w0 * qv[C0 + c]; acc[2 * ab + 1][c] += w1 * qv[C0 + c]; }
            }
        }
        __syncwarp();
    }
    const size_t M3 = pse_plane_stride(M);
    const int gz = lo[2] + 2 * rzl;
    const bool pair_ok = !(M & 1) && gz + 1 < M;                     // even M: rows start 8-byte aligned
#pragma unroll
    for (int ab = 0; ab < 4; ++ab) {
        const int gx = lo[0] + 2 * rxl + (ab >> 1), gy = lo[1] + 2 * ryl + (ab & 1);
        if (gx >= M || gy >= M || gz >= M) continue;
        const size_t o = ((size_t)gx * M + gy) * M + gz;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            float *dst = grid + (C0 + c) * M3 + o;
            if (pair_ok) *reinterpret_cast<float2 *>(dst) = make_float2(acc[2 * ab][c], acc[2 * ab + 1][c]);
            else { dst[0] = acc[2 * ab][c]; if (gz + 1 < M) dst[1] = acc[2 * ab + 1][c]; }
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

// Interpolation (a7), default path for P <= 8: one CTA per tile bin (every particle belongs to exactly one bin, so the output is
// written once, no atomics).  The (T+P-1)^3 block of the requested planes that the bin's particles can touch is staged in
// shared memory, planar, [plane][ix][iy][iz]:
//   * tiles whose block does not cross the periodic seam: ONE TMA box copy per plane (cp.async.bulk.tensor.4d on the
//     [8][M][M][M] grid array, completion on an mbarrier) issued by one thread: no staging instructions at all;
//   * seam tiles, or grids whose row pitch is not a multiple of 16 bytes (M % 4 != 0, which TMA cannot address): 4-byte
//     cp.async copies with the wrap resolved per row.
// Only the planes the product asks for are staged (3, 5 or 8), so more CTAs are resident.  Then eight lanes per particle, four
// particles per warp: a lane owns (j,k) columns of the support and walks them along x; the window values come from the
// per-particle table of pse_neighbors (no exp / sqrt here); 7-shuffle reduction leaves component gl in lane gl.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int PT> struct InterpGeom {
    static constexpr int E = T + PT - 1, EP = (E + 3) & ~3, PL = ((E * E * EP * 4 + 127) / 128 * 128) / 4;   // floats per staged plane
};

template <int PT, int C0, int NC>
__global__ void __launch_bounds__(256)
interp_planes_kernel(const __grid_constant__ CUtensorMap tmap, const int *__restrict__ pbase, const float *__restrict__ pw,
                     const int *__restrict__ tile_start, const int *__restrict__ tile_list, const float *__restrict__ grid,
                     float *__restrict__ out, int M, int nt, int accumulate, int use_tma) {
    constexpr int P = PT, E = InterpGeom<PT>::E, EP = InterpGeom<PT>::EP, PL = InterpGeom<PT>::PL, PP = (P + 3) & ~3, EE = E * EP;
    extern __shared__ __align__(128) float sm[];                    // [NC][PL]
    __shared__ __align__(8) unsigned long long bar;
    const int t = blockIdx.x, t0 = t / (nt * nt), t1 = (t / nt) % nt, t2 = t % nt;
    const int first = tile_start[t], np = tile_start[t + 1] - first;
    if (np == 0) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const bool seam = t0 * T + E > M || t1 * T + E > M || t2 * T + E > M;
    bool staged = !(use_tma && !seam);             // TMA path: every thread waits on the mbarrier itself, after its own first loads
    if (use_tma && !seam) {
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&bar)));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar)), "r"(NC * E * E * EP * 4) : "memory");
#pragma unroll
            for (int c = 0; c < NC; ++c)
                asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                             ::"r"(smem_u32(sm + c * PL)), "l"(&tmap), "r"(t2 * T), "r"(t1 * T), "r"(t0 * T), "r"(C0 + c), "r"(smem_u32(&bar))
                             : "memory");
        }
    } else {
        const size_t M3 = pse_plane_stride(M);
        // a half-warp (E <= 16) per (ix,iy) row, lanes along z; wrap by subtraction; all copies in flight at once
        const int lz = lane & 15, sub = lane >> 4;
        int gz = t2 * T + lz;
        gz -= gz >= M ? M : 0;
        for (int row = wid * 2 + sub; row < E * E; row += nw * 2) {
            const int ix = row / E, iy = row - ix * E;
            int gx = t0 * T + ix, gy = t1 * T + iy;
            gx -= gx >= M ? M : 0;
            gy -= gy >= M ? M : 0;
            if (lz < E) {
                const float *src = grid + C0 * M3 + ((size_t)gx * M + gy) * M + gz;
                float *dst = sm + row * EP + lz;
#pragma unroll
                for (int c = 0; c < NC; ++c) __pipeline_memcpy_async(dst + c * PL, src + c * M3, 4);
            }
        }
        __pipeline_commit();
        __pipeline_wait_prior(0);
        __syncthreads();
    }
    const int gl = lane & 7, grp = lane >> 3;
    for (int pi0 = wid * 4; pi0 < np; pi0 += nw * 4) {                  // uniform over the warp (shuffles inside)
        const int pi = pi0 + grp;
        const bool live = pi < np;
        const int e = first + (live ? pi : 0);                          // tile-order index: base and window rows are contiguous per tile
        const int b = pbase[e];
        const int s = tile_list[e];
        const bool mine = gl >= C0 && gl < C0 + NC;
        const float prev = (live && mine && accumulate) ? out[(size_t)s * 8 + gl] : 0.f;         // read-modify-write operand early
        const int r0 = (b & 1023) - t0 * T, r1 = ((b >> 10) & 1023) - t1 * T, r2 = ((b >> 20) & 1023) - t2 * T;   // 0..7: binned by base
        const float *wrow = pw + (size_t)e * 3 * PP;
        float wx[P];
#pragma unroll
        for (int i4 = 0; i4 < PP / 4; ++i4) {
            const float4 v = reinterpret_cast<const float4 *>(wrow)[i4];
            if (4 * i4 < P) wx[4 * i4] = v.x;
            if (4 * i4 + 1 < P) wx[4 * i4 + 1] = v.y;
            if (4 * i4 + 2 < P) wx[4 * i4 + 2] = v.z;
            if (4 * i4 + 3 < P) wx[4 * i4 + 3] = v.w;
        }
        // the window products of this lane's columns, before the staged block is needed
        constexpr int NCOL = (P * P + 7) / 8;
        float wyz[NCOL];
#pragma unroll
        for (int m = 0; m < NCOL; ++m) {
            const int jk = gl + 8 * m, j = jk / P, k = jk - j * P;
            wyz[m] = jk < P * P ? wrow[PP + j] * wrow[2 * PP + k] : 0.f;
        }
        if (!staged) {                                                  // first pass of the TMA path: the loads above are in flight
            unsigned done = 0;
            while (!done)
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                             : "=r"(done) : "r"(smem_u32(&bar)) : "memory");
            staged = true;
        }
        float acc[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[c] = 0.f;
        if (live) {
#pragma unroll
            for (int m = 0; m < NCOL; ++m) {
                const int jk = gl + 8 * m;
                if (jk < P * P) {
                    const int j = jk / P, k = jk - j * P;
                    const float *col = sm + (r0 * E + r1 + j) * EP + r2 + k;
                    float ts[NC];
#pragma unroll
                    for (int c = 0; c < NC; ++c) ts[c] = 0.f;
#pragma unroll
                    for (int i = 0; i < P; ++i)
#pragma unroll
                        for (int c = 0; c < NC; ++c) ts[c] += wx[i] * col[c * PL + i * EE];
#pragma unroll
                    for (int c = 0; c < NC; ++c) acc[c] += wyz[m] * ts[c];
                }
            }
        }
        float full[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) full[c] = (c >= C0 && c < C0 + NC) ? acc[c - C0] : 0.f;
        // 8 sums over 8 lanes in 4 + 2 + 1 shuffles: every step halves the values a lane carries
        const bool h4 = gl & 4, h2 = gl & 2, h1 = gl & 1;
        float r4[4], r2s[2];
#pragma unroll
        for (int c = 0; c < 4; ++c) r4[c] = (h4 ? full[c + 4] : full[c]) + __shfl_xor_sync(0xffffffffu, h4 ? full[c] : full[c + 4], 4);
#pragma unroll
        for (int c = 0; c < 2; ++c) r2s[c] = (h2 ? r4[c + 2] : r4[c]) + __shfl_xor_sync(0xffffffffu, h2 ? r4[c] : r4[c + 2], 2);
        const float r = (h1 ? r2s[1] : r2s[0]) + __shfl_xor_sync(0xffffffffu, h1 ? r2s[0] : r2s[1], 1);
        if (live && mine) out[(size_t)s * 8 + gl] = r + prev;
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

// a5, Brownian flavour (Eq. 75): uh = c_br sqrt((1+k^2/4xi^2)/(eta k^2)) exp(-k^2/8xi^2) / kappa(k) (I - kh kh) W(k),
// W(k) = (g_re + i g_im)/sqrt2 from the noise buffer; in the plane kz = 0 the non-canonical member of each +-k pair takes the
// conjugate of its partner's entry (reading R8) so that the C2R transform sees a Hermitian field.  The thread grid is the half
// spectrum of the FINER grid sp.M of the Brownian pass; the noise buffer is laid out on the product grid sp.Mc <= sp.M and only
// its modes carry weight (zero-padded spectrum): same field as on the product grid, interpolated with an oversampled window.
// rot != nullptr: the angular-velocity planes Omega_h = (i/2) s1 k x uh of the same random field go to rot[3][modes] (full couplet, R21).
__global__ void __launch_bounds__(256) scale_brownian_kernel(cufftComplex *spec, const float2 *__restrict__ noise, ScaleParams sp, cufftComplex *rot) {
    const int M = sp.M, Mc = sp.Mc;
    const unsigned plane = (unsigned)M * (unsigned)sp.Mh, rem = blockIdx.x * blockDim.x + threadIdx.x;
    if (rem >= plane) return;
    const int ix = (int)blockIdx.y, iy = (int)(rem / (unsigned)sp.Mh), iz = (int)(rem - (unsigned)iy * (unsigned)sp.Mh);
    const size_t nmode = (size_t)plane * M, o = (size_t)ix * plane + rem;
    const float2 zero = make_float2(0.f, 0.f);
    const int half = (M + 1) / 2, nx = ix < half ? ix : ix - M, ny = iy < half ? iy : iy - M, nz = iz;
    // modes of the product grid, its Nyquist planes and k = 0 excluded (reading R8)
    const int lim = (Mc - 1) / 2;                                      // largest |n| below the product grid's Nyquist index
    const bool live = abs(nx) <= lim && abs(ny) <= lim && nz <= lim && (nx | ny | nz) != 0;
    if (!live) {
#pragma unroll
        for (int c = 0; c < 8; ++c) spec[c * nmode + o] = zero;
        if (rot) { rot[o] = zero; rot[nmode + o] = zero; rot[2 * nmode + o] = zero; }
        return;
    }
    const float ki11 = __ldg(&sp.lat->i11), ki12 = __ldg(&sp.lat->i12), ki22 = __ldg(&sp.lat->i22);
    const float kx = sp.two_pi_over_L * (ki11 * (float)nx), ky = sp.two_pi_over_L * (ki22 * (float)ny + ki12 * (float)nx), kz = sp.two_pi_over_L * (float)nz;
    const bool canon = nz > 0 || ny > 0 || (ny == 0 && nx > 0);
    const int sx = canon ? nx : -nx, sy = canon ? ny : -ny;           // noise entry of the canonical member, product-grid indices
    const size_t cmode = (size_t)Mc * Mc * sp.Mch, src = ((size_t)(sx < 0 ? sx + Mc : sx) * Mc + (size_t)(sy < 0 ? sy + Mc : sy)) * sp.Mch + nz;
    const float sgn = canon ? 1.f : -1.f;
    float2 W[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { float2 g = noise[c * cmode + src]; W[c] = make_float2(g.x * WS_RS2, sgn * g.y * WS_RS2); }
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
    write_outputs(spec, nmode, o, s0, s1, kx, ky, kz, ux, uy, uz, PSE_OUT_U | PSE_OUT_E);
    if (rot) {
        const float h1 = 0.5f * s1;
        const float2 wx = make_float2(ky * uz.x - kz * uy.x, ky * uz.y - kz * uy.y);
        const float2 wy = make_float2(kz * ux.x - kx * uz.x, kz * ux.y - kx * uz.y);
        const float2 wz = make_float2(kx * uy.x - ky * ux.x, kx * uy.y - ky * ux.y);
        rot[o] = make_float2(-h1 * wx.y, h1 * wx.x);
        rot[nmode + o] = make_float2(-h1 * wy.y, h1 * wy.x);
        rot[2 * nmode + o] = make_float2(-h1 * wz.y, h1 * wz.x);
    }
}

}  // namespace

template <int PT, int C0, int NC>
static pse_status launch_interp_planes(pse_ctx *c, const InterpSet &g, float *d_out, bool accumulate) {
    const size_t smem = (size_t)NC * InterpGeom<PT>::PL * sizeof(float);
    interp_planes_kernel<PT, C0, NC><<<g.ntile, 256, smem, c->stream>>>(g.tmap, g.pbase, g.pw, g.tile_start, g.tile_list, g.grid,
                                                                       d_out, g.M, g.nt, accumulate ? 1 : 0, g.tma_ok ? 1 : 0);
    return PSE_OK;
}
template <int PT>
static pse_status launch_interp(pse_ctx *c, const InterpSet &g, int oplan, float *d_out, bool accumulate) {
    return oplan == 3 ? launch_interp_planes<PT, 0, 8>(c, g, d_out, accumulate)
         : oplan == 1 ? launch_interp_planes<PT, 0, 3>(c, g, d_out, accumulate) : launch_interp_planes<PT, 3, 5>(c, g, d_out, accumulate);
}
static pse_status launch_interp_any(pse_ctx *c, const InterpSet &g, int oplan, float *d_out, bool accumulate) {
    switch (g.P) {
        case 2: return launch_interp<2>(c, g, oplan, d_out, accumulate);
        case 3: return launch_interp<3>(c, g, oplan, d_out, accumulate);
        case 4: return launch_interp<4>(c, g, oplan, d_out, accumulate);
        case 5: return launch_interp<5>(c, g, oplan, d_out, accumulate);
        case 6: return launch_interp<6>(c, g, oplan, d_out, accumulate);
        case 7: return launch_interp<7>(c, g, oplan, d_out, accumulate);
        default: return launch_interp<8>(c, g, oplan, d_out, accumulate);
    }
}

// dynamic shared-memory opt-in of the interpolation kernels and the TMA descriptor of one grid array
template <int PT>
static pse_status init_interp(pse_ctx *c, InterpSet &g) {
#define PSE_INTERP_ATTR(C0, NC) CUDA_TRY(c, cudaFuncSetAttribute(interp_planes_kernel<PT, C0, NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                                                 (int)((size_t)NC * InterpGeom<PT>::PL * sizeof(float))))
    PSE_INTERP_ATTR(0, 8); PSE_INTERP_ATTR(0, 3); PSE_INTERP_ATTR(3, 5);
#undef PSE_INTERP_ATTR
    g.tma_ok = false;
    if (g.M % 4 != 0) return PSE_OK;                  // row pitch not a multiple of 16 bytes: TMA cannot address the grid
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
        cudaGetLastError();
        return PSE_OK;                                // driver without tensor maps: cp.async staging everywhere
    }
    const cuuint64_t M = (cuuint64_t)g.M;
    const cuuint64_t dims[4] = {M, M, M, 8};
    const cuuint64_t strides[3] = {M * 4, M * M * 4, (cuuint64_t)pse_plane_stride(g.M) * 4};
    const cuuint32_t box[4] = {(cuuint32_t)InterpGeom<PT>::EP, (cuuint32_t)InterpGeom<PT>::E, (cuuint32_t)InterpGeom<PT>::E, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = ((encode_fn)fn)(&g.tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, g.grid, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                       CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    g.tma_ok = (r == CUDA_SUCCESS);
    return PSE_OK;
}
static pse_status init_interp_any(pse_ctx *c, InterpSet &g) {
    switch (g.P) {
        case 2: return init_interp<2>(c, g);
        case 3: return init_interp<3>(c, g);
        case 4: return init_interp<4>(c, g);
        case 5: return init_interp<5>(c, g);
        case 6: return init_interp<6>(c, g);
        case 7: return init_interp<7>(c, g);
        case 8: return init_interp<8>(c, g);
        default: return PSE_OK;                       // wider supports take the generic kernel
    }
}

// the block-owning spread serves supports up to 8 points on grids of at least two tiles per dimension; anything else takes
// the generic gather kernel
static bool use_block_spread(const pse_ctx *c) { return c->P <= 8 && c->P != 7 && c->M >= 2 * T && c->M >= 2 * c->P; }

pse_status pse_wave_init(pse_ctx *c) {
    const int M = c->M;
    c->Mh = M / 2 + 1;
    c->Mb = std::max(M + 2, pse_choose_grid((int)std::ceil(1.18 * M)));      // finer grid of the Brownian wave pass (see pse_internal.h)
    c->Mbh = c->Mb / 2 + 1;
    c->Pb = std::min(PSE_MAXP, c->P + 1);                                      // and one more window point per dimension
    c->nt = (M + T - 1) / T; c->ntile = c->nt * c->nt * c->nt;
    const size_t M3 = pse_plane_stride(M), nmode = (size_t)M * M * c->Mh;
    CUDA_TRY(c, cudaMalloc(&c->d_grid, 8 * M3 * sizeof(float)));
    CUDA_TRY(c, cudaMalloc(&c->d_spec, 8 * nmode * sizeof(cufftComplex)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_start, (size_t)(c->ntile + 1) * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_of, (size_t)c->N * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_tile_list, (size_t)c->N * sizeof(int)));
    c->PP = (c->P + 3) & ~3;
    CUDA_TRY(c, cudaMalloc(&c->d_pbase, (size_t)c->N * sizeof(int)));
    CUDA_TRY(c, cudaMalloc(&c->d_pw, (size_t)c->N * 3 * c->PP * sizeof(float)));
    {
        InterpSet &g = c->iset;
        g.M = c->M; g.P = c->P; g.PP = c->PP; g.nt = c->nt; g.ntile = c->ntile; g.grid = c->d_grid;
        g.tile_start = c->d_tile_start; g.tile_list = c->d_tile_list; g.pbase = c->d_pbase; g.pw = c->d_pw;
        PSE_TRY(init_interp_any(c, g));
    }
    if (use_block_spread(c)) {
        // exact bound of the halves one particle can reach for this (P, M): units touched per dimension, maximised over the base
        auto max_units = [&](int UW) {
            int best = 1;
            for (int b = 0; b < M; ++b) {
                int u[4], n = 0;
                for (int i = 0; i < c->P; ++i) { const int unit = ((b + i) % M) / UW; bool seen = false; for (int q = 0; q < n; ++q) seen |= u[q] == unit; if (!seen && n < 4) u[n++] = unit; }
                best = std::max(best, n);
            }
            return best;
        };
        const int my = max_units(T);
        c->half_cap = (size_t)c->N * max_units(T / 2) * my * my;
        CUDA_TRY(c, cudaMalloc(&c->d_half_start, (size_t)(2 * c->ntile + 1) * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&c->d_half_count, (size_t)(2 * c->ntile + 1) * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&c->d_half_list, c->half_cap * sizeof(int)));
    }
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
    {   // Brownian pass: 8 planes C2R on the finer grid
        const int Mb = c->Mb, Mbh = c->Mbh;
        const size_t M3b = pse_plane_stride(Mb);
        CUDA_TRY(c, cudaMalloc(&c->d_grid_b, 8 * M3b * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&c->d_spec_b, 8 * (size_t)Mb * Mb * Mbh * sizeof(cufftComplex)));
        InterpSet &g = c->iset_b;                     // tile bins and window data of the finer grid, built on demand (pse_wave_brownian)
        g.M = Mb; g.P = c->Pb; g.PP = (c->Pb + 3) & ~3; g.nt = (Mb + T - 1) / T; g.ntile = g.nt * g.nt * g.nt; g.grid = c->d_grid_b;
        CUDA_TRY(c, cudaMalloc(&g.tile_start, (size_t)(g.ntile + 1) * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&g.tile_list, (size_t)c->N * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&g.pbase, (size_t)c->N * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&g.pw, (size_t)c->N * 3 * g.PP * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&c->d_tile_of_b, (size_t)c->N * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&c->d_tile_tmp_b, (size_t)c->N * sizeof(int)));
        CUDA_TRY(c, cudaMalloc(&c->d_tile_cnt_b, (size_t)2 * (g.ntile + 1) * sizeof(int)));
        PSE_TRY(init_interp_any(c, g));
        int nb3[3] = {Mb, Mb, Mb}, nr[3] = {Mb, Mb, Mb}, ncx[3] = {Mb, Mb, Mbh};
        size_t wb = 0;
        CUFFT_TRY(c, cufftCreate(&c->plan_c2r_b)); c->have_plan_b = true;
        CUFFT_TRY(c, cufftSetAutoAllocation(c->plan_c2r_b, 0));
        CUFFT_TRY(c, cufftMakePlanMany(c->plan_c2r_b, 3, nb3, ncx, 1, Mb * Mb * Mbh, nr, 1, (int)M3b, CUFFT_C2R, 8, &wb));
        w = std::max(w, wb);
    }
    if (w) CUDA_TRY(c, cudaMalloc(&c->d_fft_work, w));
    CUFFT_TRY(c, cufftSetWorkArea(c->plan_c2r_b, c->d_fft_work)); CUFFT_TRY(c, cufftSetStream(c->plan_c2r_b, c->stream));
    for (int i = 0; i < 3; ++i) {
        CUFFT_TRY(c, cufftSetWorkArea(c->plan_r2c[i], c->d_fft_work)); CUFFT_TRY(c, cufftSetWorkArea(c->plan_c2r[i], c->d_fft_work));
        CUFFT_TRY(c, cufftSetStream(c->plan_r2c[i], c->stream)); CUFFT_TRY(c, cufftSetStream(c->plan_c2r[i], c->stream));
    }
    return PSE_OK;
}

void pse_wave_set_stream(pse_ctx *c, cudaStream_t st) {
    for (int i = 0; i < c->nplans; ++i) { cufftSetStream(c->plan_r2c[i], st); cufftSetStream(c->plan_c2r[i], st); }
    if (c->have_plan_b) cufftSetStream(c->plan_c2r_b, st);
    if (c->have_plan_rot_b) cufftSetStream(c->plan_c2r_rot_b, st);
}

void pse_wave_free(pse_ctx *c) {
    for (int i = 0; i < c->nplans; ++i) { cufftDestroy(c->plan_r2c[i]); cufftDestroy(c->plan_c2r[i]); }
    if (c->have_plan_b) cufftDestroy(c->plan_c2r_b);
    if (c->have_plan_rot_b) cufftDestroy(c->plan_c2r_rot_b);
    cudaFree(c->d_grid_b); cudaFree(c->d_spec_b); cudaFree(c->d_spec_rot_b);
    cudaFree(c->iset_b.tile_start); cudaFree(c->iset_b.tile_list); cudaFree(c->iset_b.pbase); cudaFree(c->iset_b.pw);
    cudaFree(c->d_tile_of_b); cudaFree(c->d_tile_tmp_b); cudaFree(c->d_tile_cnt_b);
    cudaFree(c->d_grid); cudaFree(c->d_spec); cudaFree(c->d_fft_work);
    cudaFree(c->d_tile_start); cudaFree(c->d_tile_of); cudaFree(c->d_tile_list); cudaFree(c->d_pbase); cudaFree(c->d_pw);
    cudaFree(c->d_half_start); cudaFree(c->d_half_count); cudaFree(c->d_half_list);
}

// Tile bins: counted in wrap_and_bin, scanned with the cell counts, scattered in gather_positions (neighbors.cu);
// what is left is the deterministic order inside every tile.
pse_status pse_tile_bins(pse_ctx *c) {
    return pse_rank_sort(c, c->d_tile_start, c->ntile, c->d_tile_tmp, c->d_tile_list);
}

static pse_status launch_particle_window(pse_ctx *c, const InterpSet &g, double wa_d, double wb_d) {
    const float4 *pos = c->d_pos;
    float4 *pw4 = reinterpret_cast<float4 *>(g.pw);
    const float ih = (float)(g.M / c->L), wa = (float)wa_d, wb = (float)wb_d;
    const int nb = (c->N + 127) / 128;
    switch (g.PP) {
        case 4: particle_window_kernel<4><<<nb, 128, 0, c->stream>>>(pos, g.tile_list, c->N, g.M, g.P, ih, wa, wb, g.pbase, pw4); break;
        case 8: particle_window_kernel<8><<<nb, 128, 0, c->stream>>>(pos, g.tile_list, c->N, g.M, g.P, ih, wa, wb, g.pbase, pw4); break;
        case 12: particle_window_kernel<12><<<nb, 128, 0, c->stream>>>(pos, g.tile_list, c->N, g.M, g.P, ih, wa, wb, g.pbase, pw4); break;
        default: particle_window_kernel<16><<<nb, 128, 0, c->stream>>>(pos, g.tile_list, c->N, g.M, g.P, ih, wa, wb, g.pbase, pw4); break;
    }
    KERNEL_CHECK(c);
    return PSE_OK;
}

// tile bins and window data of the finer grid for the current (cell-sorted) positions; no-op if they are current
static pse_status ensure_fine_bins(pse_ctx *c) {
    if (c->fine_bins_valid) return PSE_OK;
    InterpSet &g = c->iset_b;
    const int N = c->N, nb = (N + 255) / 256;
    int *count = c->d_tile_cnt_b, *fill = c->d_tile_cnt_b + g.ntile + 1;
    CUDA_TRY(c, cudaMemsetAsync(c->d_tile_cnt_b, 0, (size_t)2 * (g.ntile + 1) * sizeof(int), c->stream));
    fine_bin_count<<<nb, 256, 0, c->stream>>>(c->d_pos, N, (float)(g.M / c->L), g.M, g.P, g.nt, c->d_tile_of_b, count); KERNEL_CHECK(c);
    PSE_TRY(pse_scan_i32(c, count, g.tile_start, (size_t)g.ntile));
    fine_bin_scatter<<<nb, 256, 0, c->stream>>>(c->d_tile_of_b, N, g.tile_start, fill, c->d_tile_tmp_b); KERNEL_CHECK(c);
    PSE_TRY(pse_rank_sort(c, g.tile_start, g.ntile, c->d_tile_tmp_b, g.tile_list));
    PSE_TRY(launch_particle_window(c, g, c->win_a_b, c->win_b_b));
    c->fine_bins_valid = true;
    return PSE_OK;
}

pse_status pse_particle_windows(pse_ctx *c) {
    c->fine_bins_valid = false;                                      // new positions
    PSE_TRY(launch_particle_window(c, c->iset, c->win_a, c->win_b));
    if (!use_block_spread(c)) return PSE_OK;
    // lists of the particles that reach every half tile: one pass, segments reserved on a cursor (cleared with the bin counters)
    const int nhalf = 2 * c->ntile;
    half_lists_kernel<<<(nhalf + HL_WARPS - 1) / HL_WARPS, HL_WARPS * 32, 0, c->stream>>>(c->d_pbase, c->d_tile_start, c->M, c->P, c->nt, nhalf,
                                                                                        c->d_half_start, c->d_half_count, c->d_half_list, c->d_half_cursor);
    KERNEL_CHECK(c);
    return PSE_OK;
}

template <int P>
static void launch_spread_blocks(pse_ctx *c, int plan, const float4 *in4) {
    if (plan == 0) spread_blocks_kernel<P, 0, 8><<<c->ntile, 64, 0, c->stream>>>(c->d_pbase, c->d_pw, c->d_tile_list, in4, c->d_half_start, c->d_half_count, c->d_half_list, c->d_grid, c->M, c->nt);
    else if (plan == 1) spread_blocks_kernel<P, 0, 3><<<c->ntile, 64, 0, c->stream>>>(c->d_pbase, c->d_pw, c->d_tile_list, in4, c->d_half_start, c->d_half_count, c->d_half_list, c->d_grid, c->M, c->nt);
    else spread_blocks_kernel<P, 3, 5><<<c->ntile, 64, 0, c->stream>>>(c->d_pbase, c->d_pw, c->d_tile_list, in4, c->d_half_start, c->d_half_count, c->d_half_list, c->d_grid, c->M, c->nt);
}

// plane range of a 2-bit component mask (bit 0: planes 0-2, bit 1: planes 3-7): plan index and first plane
static inline void plane_range(int bits, int &plan, int &first) {
    plan = bits == 3 ? 0 : bits; first = bits == 2 ? 3 : 0;
}

// interpolation of the planes of one output plan from c->d_grid (oplan bit 0: planes 0-2, bit 1: planes 3-7)
pse_status pse_wave_interp(pse_ctx *c, float *d_out, bool accumulate, int oplan) {
    ScopedPhase ph(c, PSE_T_INTERP);
    const int TB = 256;
    if (c->P <= 8) {
        PSE_TRY(launch_interp_any(c, c->iset, oplan, d_out, accumulate));
    } else {
        interp_kernel<<<(unsigned)(((size_t)c->N * 32 + TB - 1) / TB), TB, 0, c->stream>>>(
            c->d_pos, c->d_tile_list, c->d_grid, reinterpret_cast<float4 *>(d_out), c->N, c->M, c->P, (float)(1.0 / c->h),
            (float)c->win_a, (float)c->win_b, accumulate ? 1 : 0, oplan << 2);
    }
    KERNEL_CHECK(c);
    return PSE_OK;
}

static pse_status inverse_and_interpolate(pse_ctx *c, float *d_out, bool accumulate, int mode = PSE_MODE_ALL) {
    {
        ScopedPhase ph(c, PSE_T_FFT_INV);
        int plan, first;
        plane_range((mode >> 2) & 3, plan, first);
        const size_t M3 = pse_plane_stride(c->M), nmode = (size_t)c->M * c->M * c->Mh;
        CUFFT_TRY(c, cufftExecC2R(c->plan_c2r[plan], c->d_spec + first * nmode, c->d_grid + first * M3)); c->launches++;
    }
    return pse_wave_interp(c, d_out, accumulate, (mode >> 2) & 3);
}

// spread of the planes of one input plan (0: all 8, 1: planes 0-2, 2: planes 3-7) of the packed vector d_in into c->d_grid
pse_status pse_wave_spread(pse_ctx *c, const float *d_in, int plan) {
    ScopedPhase ph(c, PSE_T_SPREAD);
    const float4 *in4 = reinterpret_cast<const float4 *>(d_in);
    const float ih = (float)(1.0 / c->h), wa = (float)c->win_a, wb = (float)c->win_b;
    if (use_block_spread(c)) {
        switch (c->P) {
            case 2: launch_spread_blocks<2>(c, plan, in4); break;
            case 3: launch_spread_blocks<3>(c, plan, in4); break;
            case 4: launch_spread_blocks<4>(c, plan, in4); break;
            case 5: launch_spread_blocks<5>(c, plan, in4); break;
            case 6: launch_spread_blocks<6>(c, plan, in4); break;
            default: launch_spread_blocks<8>(c, plan, in4); break;
        }
    } else if (plan == 0) spread_kernel<0, 8><<<c->ntile, SPREAD_THREADS, 0, c->stream>>>(c->d_pos, in4, c->d_tile_start, c->d_tile_list, c->d_grid, c->M, c->P, c->nt, ih, wa, wb);
    else if (plan == 1) spread_kernel<0, 3><<<c->ntile, SPREAD_THREADS, 0, c->stream>>>(c->d_pos, in4, c->d_tile_start, c->d_tile_list, c->d_grid, c->M, c->P, c->nt, ih, wa, wb);
    else spread_kernel<3, 5><<<c->ntile, SPREAD_THREADS, 0, c->stream>>>(c->d_pos, in4, c->d_tile_start, c->d_tile_list, c->d_grid, c->M, c->P, c->nt, ih, wa, wb);
    KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_wave_apply(pse_ctx *c, const float *d_in, float *d_out, bool accumulate, int mode) {
    const size_t nmode = (size_t)c->M * c->M * c->Mh, M3 = pse_plane_stride(c->M);
    if (!(mode & (PSE_IN_F | PSE_IN_S)) || !(mode & (PSE_OUT_U | PSE_OUT_E))) { c->err = "pse_wave_apply: empty component mask"; return PSE_EINVAL; }
    int plan, first;
    plane_range(mode & 3, plan, first);
    PSE_TRY(pse_wave_spread(c, d_in, plan));
    { ScopedPhase ph(c, PSE_T_FFT_FWD); CUFFT_TRY(c, cufftExecR2C(c->plan_r2c[plan], c->d_grid + first * M3, c->d_spec + first * nmode)); c->launches++; }
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        scale_kernel<<<dim3((unsigned)((c->M * c->Mh + 255) / 256), (unsigned)c->M), 256, 0, c->stream>>>(c->d_spec, make_scale_params(c, mode)); KERNEL_CHECK(c);
    }
    return inverse_and_interpolate(c, d_out, accumulate, mode);
}

// d_outW != nullptr (full couplet): the angular velocities of the same field are ADDED to slots 0-2 of the packed vector d_outW;
// three more spectra and a 3-plane C2R plan on the finer grid are made by the first such call.
pse_status pse_wave_brownian(pse_ctx *c, const float *d_noise_wave, float *d_out, bool accumulate, float *d_outW) {
    if (c->noise_pending) { CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->ev_noise, 0)); c->noise_pending = false; }
    const int Mb = c->Mb;
    if (d_outW && !c->d_spec_rot_b) {
        const size_t M3b = pse_plane_stride(Mb);
        if (cudaMalloc(&c->d_spec_rot_b, 3 * (size_t)Mb * Mb * c->Mbh * sizeof(cufftComplex)) != cudaSuccess) {
            cudaGetLastError(); c->d_spec_rot_b = nullptr; c->err = "out of memory (angular-velocity spectra of the Brownian pass)"; return PSE_ENOMEM;
        }
        int nb3[3] = {Mb, Mb, Mb}, nr[3] = {Mb, Mb, Mb}, ncx[3] = {Mb, Mb, c->Mbh};
        CUFFT_TRY(c, cufftPlanMany(&c->plan_c2r_rot_b, 3, nb3, ncx, 1, Mb * Mb * c->Mbh, nr, 1, (int)M3b, CUFFT_C2R, 3)); c->have_plan_rot_b = true;
        CUFFT_TRY(c, cufftSetStream(c->plan_c2r_rot_b, c->stream));
    }
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        ScaleParams sp = make_scale_params(c);
        sp.M = Mb; sp.Mh = c->Mbh; sp.dec = c->d_dec_b;               // thread grid and window table of the finer grid; noise on (Mc, Mch)
        scale_brownian_kernel<<<dim3((unsigned)((Mb * c->Mbh + 255) / 256), (unsigned)Mb), 256, 0, c->stream>>>(
            c->d_spec_b, reinterpret_cast<const float2 *>(d_noise_wave), sp, d_outW ? c->d_spec_rot_b : nullptr);
        KERNEL_CHECK(c);
    }
    { ScopedPhase ph(c, PSE_T_FFT_INV); CUFFT_TRY(c, cufftExecC2R(c->plan_c2r_b, c->d_spec_b, c->d_grid_b)); c->launches++; }
    ScopedPhase ph(c, PSE_T_INTERP);
    if (c->Pb <= 8) {
        PSE_TRY(ensure_fine_bins(c));
        PSE_TRY(launch_interp_any(c, c->iset_b, 3, d_out, accumulate));
    } else {
        const int TB = 256;
        interp_kernel<<<(unsigned)(((size_t)c->N * 32 + TB - 1) / TB), TB, 0, c->stream>>>(
            c->d_pos, c->d_tile_list, c->d_grid_b, reinterpret_cast<float4 *>(d_out), c->N, Mb, c->Pb, (float)(Mb / c->L),
            (float)c->win_a_b, (float)c->win_b_b, accumulate ? 1 : 0, PSE_MODE_ALL);
    }
    KERNEL_CHECK(c);
    if (!d_outW) return PSE_OK;
    // the three angular-velocity planes pass through planes 0-2 of the finer grid array
    CUFFT_TRY(c, cufftExecC2R(c->plan_c2r_rot_b, c->d_spec_rot_b, c->d_grid_b)); c->launches++;
    if (c->Pb <= 8) {
        PSE_TRY(launch_interp_any(c, c->iset_b, 1, d_outW, true));
    } else {
        const int TB = 256;
        interp_kernel<<<(unsigned)(((size_t)c->N * 32 + TB - 1) / TB), TB, 0, c->stream>>>(
            c->d_pos, c->d_tile_list, c->d_grid_b, reinterpret_cast<float4 *>(d_outW), c->N, Mb, c->Pb, (float)(Mb / c->L),
            (float)c->win_a_b, (float)c->win_b_b, 1, PSE_OUT_U);
    }
    KERNEL_CHECK(c);
    return PSE_OK;
}

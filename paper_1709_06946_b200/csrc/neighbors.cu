// Cell list + full neighbour list (step a1; "linked-cell lists ... sub-cells of size r_cut").
//
// Design (sm_100a, not a translation of HOOMD's lists): counting sort of particles by cell (deterministic: each cell's
// members are re-sorted by original index), positions gathered into cell order, then ONE pass with a CTA per cell
// (neighbor_build_cell): the <= 18 contiguous candidate runs of the cell are staged in shared memory, every
// (particle, candidate) pair is tested once with the hits kept as bit masks, the cell reserves its segment of the index
// array with one atomicAdd on a cursor and expands the masks into it.  Cells too large for the mask store take a two-pass
// count / scan / fill path (neighbor_sweep_cell), remembered per context.  The in/out decision is taken in fp32 with the
// exact operation order of DESIGN.md reading R16 (no FMA contraction), so the sets are bit-identical to the oracle's.
// The host never waits for the build: the list size and the overflow / fallback flags come back asynchronously and are
// examined at the next point where the stream is synchronised anyway (pse_neighbors_settle).
#include <cmath>
#include "pse_internal.h"

namespace {

constexpr int SCAN_ITEMS = 8, SCAN_THREADS = 256, SCAN_CHUNK = SCAN_ITEMS * SCAN_THREADS;

__device__ __forceinline__ unsigned long long block_exclusive_scan(unsigned long long v, unsigned long long *total) {
    __shared__ unsigned long long warp_sums[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned long long inc = v;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        unsigned long long s = (lane < (blockDim.x >> 5)) ? warp_sums[lane] : 0ull, si = s;
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        warp_sums[lane] = si - s;
        if (lane == 31 && total) *total = si;
    }
    __syncthreads();
    unsigned long long r = warp_sums[wid] + inc - v;
    __syncthreads();
    return r;
}

__global__ void scan_block_sums(const int *in, size_t n, unsigned long long *bsum) {
    __shared__ unsigned long long tot;
    size_t base = (size_t)blockIdx.x * SCAN_CHUNK + (size_t)threadIdx.x * SCAN_ITEMS;
    unsigned long long s = 0;
    for (int i = 0; i < SCAN_ITEMS; ++i) if (base + i < n) s += (unsigned long long)in[base + i];
    block_exclusive_scan(s, &tot);
    if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

__global__ void scan_of_sums(unsigned long long *bsum, size_t nb) {      // single block, in place, exclusive
    __shared__ unsigned long long tot, carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (size_t lo = 0; lo < nb; lo += blockDim.x) {
        size_t i = lo + threadIdx.x;
        unsigned long long v = i < nb ? bsum[i] : 0ull;
        unsigned long long e = block_exclusive_scan(v, &tot);
        if (i < nb) bsum[i] = carry + e;
        __syncthreads();
        if (threadIdx.x == 0) carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) bsum[nb] = carry;
}

template <typename OutT>
__global__ void scan_apply(const int *in, size_t n, const unsigned long long *bsum, size_t nb, OutT *out) {
    size_t base = (size_t)blockIdx.x * SCAN_CHUNK + (size_t)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS]; unsigned long long s = 0;
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = (base + i < n) ? in[base + i] : 0; s += (unsigned long long)v[i]; }
    unsigned long long e = block_exclusive_scan(s, nullptr) + bsum[blockIdx.x];
    for (int i = 0; i < SCAN_ITEMS; ++i) { if (base + i < n) out[base + i] = (OutT)e; e += (unsigned long long)v[i]; }
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = (OutT)bsum[nb];
}

// whole scan in one CTA for short inputs (cell and tile counts: a few thousand entries): one launch instead of three
constexpr int SCAN1_THREADS = 1024, SCAN1_MAX = 1 << 14;
template <typename OutT>
__global__ void __launch_bounds__(SCAN1_THREADS) scan_single_cta(const int *in, int n, OutT *out) {
    __shared__ unsigned long long tot;
    const int per = (n + SCAN1_THREADS - 1) / SCAN1_THREADS, lo = threadIdx.x * per, hi = min(n, lo + per);
    unsigned long long s = 0;
    for (int i = lo; i < hi; ++i) s += (unsigned long long)in[i];
    unsigned long long e = block_exclusive_scan(s, &tot);
    for (int i = lo; i < hi; ++i) { out[i] = (OutT)e; e += (unsigned long long)in[i]; }
    if (threadIdx.x == 0) out[n] = (OutT)tot;
}

// two short scans in one launch (cell counts and tile counts)
__global__ void __launch_bounds__(SCAN1_THREADS) scan_two_ctas(const int *in0, int n0, int *out0, const int *in1, int n1, int *out1) {
    __shared__ unsigned long long tot;
    const int *in = blockIdx.x ? in1 : in0;
    int *out = blockIdx.x ? out1 : out0;
    const int n = blockIdx.x ? n1 : n0;
    const int per = (n + SCAN1_THREADS - 1) / SCAN1_THREADS, lo = threadIdx.x * per, hi = min(n, lo + per);
    unsigned long long s = 0;
    for (int i = lo; i < hi; ++i) s += (unsigned long long)in[i];
    unsigned long long e = block_exclusive_scan(s, &tot);
    for (int i = lo; i < hi; ++i) { out[i] = (int)e; e += (unsigned long long)in[i]; }
    if (threadIdx.x == 0) out[n] = (int)tot;
}

template <typename OutT>
pse_status scan_impl(pse_ctx *c, const int *d_in, OutT *d_out, size_t n) {
    if (n <= (size_t)SCAN1_MAX && (const void *)d_in != (const void *)d_out) {
        scan_single_cta<OutT><<<1, SCAN1_THREADS, 0, c->stream>>>(d_in, (int)n, d_out); KERNEL_CHECK(c);
        return PSE_OK;
    }
    size_t nb = (n + SCAN_CHUNK - 1) / SCAN_CHUNK;
    if (nb == 0) nb = 1;
    if (c->scan_tmp_n < nb + 1) {
        if (c->d_scan_tmp) cudaFree(c->d_scan_tmp);
        CUDA_TRY(c, cudaMalloc(&c->d_scan_tmp, (nb + 1) * sizeof(unsigned long long)));
        c->scan_tmp_n = nb + 1;
    }
    scan_block_sums<<<(unsigned)nb, SCAN_THREADS, 0, c->stream>>>(d_in, n, c->d_scan_tmp); KERNEL_CHECK(c);
    scan_of_sums<<<1, 1024, 0, c->stream>>>(c->d_scan_tmp, nb); KERNEL_CHECK(c);
    scan_apply<OutT><<<(unsigned)nb, SCAN_THREADS, 0, c->stream>>>(d_in, n, c->d_scan_tmp, nb, d_out); KERNEL_CHECK(c);
    return PSE_OK;
}

// ---- R16 arithmetic: every operation individually rounded, no contraction ----
__device__ __forceinline__ float wrap_coord(float x, float L, float invL) {
    float w = __fsub_rn(x, __fmul_rn(L, floorf(__fmul_rn(x, invL))));
    return (w >= L || w < 0.f) ? 0.f : w;
}
__device__ __forceinline__ float min_image(float d, float L, float invL) {
    return __fsub_rn(d, __fmul_rn(L, rintf(__fmul_rn(d, invL))));
}
// a, b: lattice coordinates; the physical separation is r = A d (reading R22).  On the cube (a11 = a22 = 1, a12 = 0) the
// extra products and the sum are exact, so the value is bit for bit that of the plain R16 form.
__device__ __forceinline__ float dist2(float4 a, float4 b, float L, float invL, Lat lat) {
    float dx = min_image(__fsub_rn(a.x, b.x), L, invL);
    float dy = min_image(__fsub_rn(a.y, b.y), L, invL);
    float dz = min_image(__fsub_rn(a.z, b.z), L, invL);
    const float rx = __fadd_rn(__fmul_rn(lat.a11, dx), __fmul_rn(lat.a12, dy)), ry = __fmul_rn(lat.a22, dy);
    return __fadd_rn(__fadd_rn(__fmul_rn(rx, rx), __fmul_rn(ry, ry)), __fmul_rn(dz, dz));
}

__global__ void wrap_and_bin(const float4 *pos, int N, float L, float invL, Cells nc, float3 cell_inv,
                             float4 *posw, int *cell_of, int *cell_count, float inv_h, int M, int P, int nt, int *tile_of, int *tile_count, const Lat *__restrict__ latp) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const Lat lat = *latp;
    float4 p = pos[i];
    p.x = __fadd_rn(__fmul_rn(lat.i11, p.x), __fmul_rn(lat.i12, p.y)); p.y = __fmul_rn(lat.i22, p.y);     // s = A^-1 x (exact on the cube)
    p.x = wrap_coord(p.x, L, invL); p.y = wrap_coord(p.y, L, invL); p.z = wrap_coord(p.z, L, invL); p.w = 0.f;
    posw[i] = p;
    int cx = min(nc.x - 1, (int)(p.x * cell_inv.x)), cy = min(nc.y - 1, (int)(p.y * cell_inv.y)), cz = min(nc.z - 1, (int)(p.z * cell_inv.z));
    int cell = (cx * nc.y + cy) * nc.z + cz;
    cell_of[i] = cell;
    atomicAdd(&cell_count[cell], 1);
    const int t = pse_tile_of(p, inv_h, M, P, nt);              // spread / interpolate tile bin of the same particle
    tile_of[i] = t;
    atomicAdd(&tile_count[t], 1);
}

__global__ void scatter_to_cells(const int *cell_of, int N, const int *cell_start, int *cell_fill, int *order) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int cell = cell_of[i];
    order[cell_start[cell] + atomicAdd(&cell_fill[cell], 1)] = i;
}

// Deterministic order inside every segment (cell or tile): warp per segment, rank sort out of place.
// rank_i = #{j : v_j < v_i} (values are distinct particle indices), n^2/32 comparisons per warp.
__global__ void rank_sort_segments(const int *__restrict__ seg_start, int nseg, const int *__restrict__ in, int *__restrict__ out) {
    int seg = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (seg >= nseg) return;
    const int lo = seg_start[seg], n = seg_start[seg + 1] - lo;
    for (int i0 = 0; i0 < n; i0 += 32) {
        const int i = i0 + lane;
        const int v = i < n ? in[lo + i] : 0x7fffffff;
        int rank = 0;
        for (int j = 0; j < n; ++j) rank += (in[lo + j] < v);
        if (i < n) out[lo + rank] = v;
    }
}

// positions into cell-sorted numbering; the sorted index is appended to the particle's tile bin on the way
__global__ void gather_positions(const float4 *posw, const int *order, int N, float4 *pos_sorted, const int *tile_of, const int *tile_start,
                                 int *tile_fill, int *tile_list) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const int o = order[s], t = tile_of[o];
    pos_sorted[s] = posw[o];
    tile_list[tile_start[t] + atomicAdd(&tile_fill[t], 1)] = s;
}

// Neighbour sweep, CTA per cell, two passes (fallback for oversized cells).  The candidates of a cell are the same for all of its particles:
// up to 18 contiguous runs of the cell-sorted order (9 (x,y) columns, z-1..z+1 contiguous, split where z wraps).
// They are staged once in shared memory in chunks of NS_CHUNK; each warp then takes particles of the cell and tests
// 32 staged candidates per iteration with full lanes.  FILL=false accumulates counts, FILL=true writes the CSR
// list in candidate order (deterministic).  Running per-particle positions live in `cursor` (global, zeroed).
constexpr int NS_CHUNK = 1024, NS_THREADS = 128;

template <bool FILL>
__global__ void __launch_bounds__(NS_THREADS) neighbor_sweep_cell(const float4 *__restrict__ pos, const int *__restrict__ cell_start,
                                                                   Cells nc, float L, float invL, float rc2, int *__restrict__ cursor,
                                                                   const unsigned long long *__restrict__ off, int *__restrict__ idx, const Lat *__restrict__ latp) {
    __shared__ float4 cpos[NS_CHUNK];
    __shared__ int run_lo[18], run_cum[19];
    const Lat lat = *latp;
    const int cell = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int first = cell_start[cell], np = cell_start[cell + 1] - first;
    if (np == 0) return;
    const int cz = cell % nc.z, cy = (cell / nc.z) % nc.y, cx = cell / (nc.y * nc.z);
    const int spanx = nc.x >= 3 ? 3 : nc.x, spany = nc.y >= 3 ? 3 : nc.y;
    if (tid < 32) {
        // lane r < 2*spanx*spany describes run r: column (r>>1), part (r&1)
        int lo = 0, len = 0;
        const int col_i = lane >> 1, part = lane & 1;
        if (col_i < spanx * spany) {
            int ccx = col_i / spany, ccy = col_i % spany;
            if (nc.x >= 3) { ccx = cx + ccx - 1; ccx += ccx < 0 ? nc.x : 0; ccx -= ccx >= nc.x ? nc.x : 0; }
            if (nc.y >= 3) { ccy = cy + ccy - 1; ccy += ccy < 0 ? nc.y : 0; ccy -= ccy >= nc.y ? nc.y : 0; }
            const int col = (ccx * nc.y + ccy) * nc.z;
            const int z0 = nc.z >= 3 ? cz - 1 : 0, z1 = nc.z >= 3 ? cz + 1 : nc.z - 1;
            int a0, a1, b0 = 0, b1 = 0;                    // run A = cells [a0,a1), run B = cells [b0,b1)
            if (z0 < 0) { a0 = 0; a1 = z1 + 1; b0 = nc.z - 1; b1 = nc.z; }
            else if (z1 >= nc.z) { a0 = 0; a1 = 1; b0 = z0; b1 = nc.z; }
            else { a0 = z0; a1 = z1 + 1; }
            const int c0 = part ? b0 : a0, c1 = part ? b1 : a1;
            lo = cell_start[col + c0]; len = cell_start[col + c1] - lo;
        }
        int inc = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
        if (lane < 18) { run_lo[lane] = lo; run_cum[lane] = inc - len; }
        if (lane == 17) run_cum[18] = inc;
    }
    __syncthreads();
    const int total = run_cum[18];
    for (int c0 = 0; c0 < total; c0 += NS_CHUNK) {
        const int nchunk = min(NS_CHUNK, total - c0);
        for (int c = tid; c < nchunk; c += NS_THREADS) {
            const int g = c0 + c;
            int r = 0;
            while (run_cum[r + 1] <= g) ++r;
            const int j = run_lo[r] + g - run_cum[r];
            float4 q = pos[j];
            q.w = __int_as_float(j);
            cpos[c] = q;
        }
        __syncthreads();
        for (int pi = wid; pi < np; pi += NS_THREADS / 32) {
            const int s = first + pi;
            const float4 p = pos[s];
            int found = (c0 == 0) ? 0 : cursor[s];
            const unsigned long long base = FILL ? off[s] : 0ull;
            for (int c = lane; c < nchunk + lane; c += 32) {        // all lanes take the same number of trips
                bool in = false;
                int j = -1;
                if (c < nchunk) {
                    const float4 q = cpos[c];
                    j = __float_as_int(q.w);
                    in = (j != s) && dist2(p, q, L, invL, lat) < rc2;
                }
                const unsigned m = __ballot_sync(0xffffffffu, in);
                if (FILL && in) idx[base + found + __popc(m & ((1u << lane) - 1))] = j;
                found += __popc(m);
                if (c - lane + 32 >= nchunk) break;
            }
            if (lane == 0) cursor[s] = found;
        }
        __syncthreads();
    }
}

// Single-pass neighbour build, CTA per cell (default path).  Pass A tests every (particle, candidate) pair once and
// keeps the 32-bit hit masks in shared memory; the cell's total is then reserved with ONE atomicAdd on a global
// cursor, and pass B expands the masks into the reserved segment.  A particle's list is deterministic (candidate
// order); only the placement of whole cells in the index array depends on scheduling, which no consumer sees
// (they go through off[s], count[s]).  Cells too large for the mask store (> NB_MAXP particles or > NS_CHUNK
// candidates) set *fallback and are handled by the two-pass kernels above.
constexpr int NB_MAXP = 64, NB_WORDS = NS_CHUNK / 32, NB_PB = 4;

template <bool DEF>                                           // DEF: deformed lattice, the screened separation is mapped by A as well
__global__ void __launch_bounds__(NS_THREADS) neighbor_build_cell(const float4 *__restrict__ pos, const int *__restrict__ cell_start, Cells nc,
                                                                   float L, float invL, float rc2, float band0, int *__restrict__ count,
                                                                   unsigned long long *__restrict__ off, int *__restrict__ idx,
                                                                   unsigned long long cap, unsigned long long *__restrict__ cursor,
                                                                   int *__restrict__ fallback, const Lat *__restrict__ latp) {
    // the lattice is read from device memory so that a captured step stays valid while the strain advances (pse_set_lattice)
    const Lat lat = DEF ? *latp : Lat{1.f, 0.f, 1.f, 1.f, 0.f, 1.f};
    const float band = DEF ? band0 * 4.f * (fabsf(lat.a11) + fabsf(lat.a12) + fabsf(lat.a22)) : band0;
    __shared__ float4 cpos[NS_CHUNK];
    __shared__ unsigned masks[NB_MAXP][NB_WORDS];
    __shared__ int cnt[NB_MAXP], loc[NB_MAXP];
    __shared__ int run_lo[18], run_cum[19];
    __shared__ unsigned long long base_s;
    __shared__ int self_s;
    const int cell = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int first = cell_start[cell], np = cell_start[cell + 1] - first;
    if (np == 0) return;
    const int cz = cell % nc.z, cy = (cell / nc.z) % nc.y, cx = cell / (nc.y * nc.z);
    const int spanx = nc.x >= 3 ? 3 : nc.x, spany = nc.y >= 3 ? 3 : nc.y;
    if (tid < 32) {
        int lo = 0, len = 0;
        const int col_i = lane >> 1, part = lane & 1;
        if (col_i < spanx * spany) {
            int ccx = col_i / spany, ccy = col_i % spany;
            if (nc.x >= 3) { ccx = cx + ccx - 1; ccx += ccx < 0 ? nc.x : 0; ccx -= ccx >= nc.x ? nc.x : 0; }
            if (nc.y >= 3) { ccy = cy + ccy - 1; ccy += ccy < 0 ? nc.y : 0; ccy -= ccy >= nc.y ? nc.y : 0; }
            const int col = (ccx * nc.y + ccy) * nc.z;
            const int z0 = nc.z >= 3 ? cz - 1 : 0, z1 = nc.z >= 3 ? cz + 1 : nc.z - 1;
            int a0, a1, b0 = 0, b1 = 0;
            if (z0 < 0) { a0 = 0; a1 = z1 + 1; b0 = nc.z - 1; b1 = nc.z; }
            else if (z1 >= nc.z) { a0 = 0; a1 = 1; b0 = z0; b1 = nc.z; }
            else { a0 = z0; a1 = z1 + 1; }
            const int c0 = part ? b0 : a0, c1 = part ? b1 : a1;
            lo = cell_start[col + c0]; len = cell_start[col + c1] - lo;
        }
        int inc = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
        if (lane < 18) { run_lo[lane] = lo; run_cum[lane] = inc - len; }
        if (lane == 17) run_cum[18] = inc;
    }
    __syncthreads();
    const int total = run_cum[18];
    if (np > NB_MAXP || total > NS_CHUNK) {                 // uniform over the CTA
        if (tid == 0) atomicExch(fallback, 1);
        return;
    }
    // Screening: with >= 5 cells per edge every candidate has one periodic image within reach of the whole cell, so it is
    // staged already shifted to that image and the test is a plain difference.  The decision itself stays the R16
    // arithmetic: whenever the screened d^2 falls within `band` of r_c^2 (far wider than the rounding difference between
    // the two forms) the pair is re-evaluated with dist2 on the unshifted position.
    const bool fast = nc.x >= 5 && nc.y >= 5 && nc.z >= 5;
    const float mx = ((float)cx + 0.5f) * (L / (float)nc.x), my = ((float)cy + 0.5f) * (L / (float)nc.y), mz = ((float)cz + 0.5f) * (L / (float)nc.z);
    const int nwords = (total + 31) >> 5;
    for (int r = wid; r < 18; r += NS_THREADS / 32) {            // staging: a warp per run, no search for the run of a candidate
        const int lo = run_lo[r], c0 = run_cum[r], len = run_cum[r + 1] - c0;
        if (first >= lo && first < lo + len && lane == 0) self_s = c0 + first - lo;     // where the cell's own particles sit
        for (int i = lane; i < len; i += 32) {
            float4 q = pos[lo + i];
            if (fast) { q.x -= L * rintf((q.x - mx) * invL); q.y -= L * rintf((q.y - my) * invL); q.z -= L * rintf((q.z - mz) * invL); }
            q.w = __int_as_float(lo + i);
            cpos[c0 + i] = q;
        }
    }
    // padding of the last word: infinitely far, index -1 (d^2 = inf: neither a hit nor inside the band)
    if (tid < nwords * 32 - total) cpos[total + tid] = make_float4(3e37f, 3e37f, 3e37f, __int_as_float(-1));
    __syncthreads();
    const int self0 = self_s;
    // pass A: distance tests, masks, counts.  A warp takes NB_PB particles at a time so that one staged candidate
    // (one LDS.128 per lane) is tested against all of them; the particle's own entry (d^2 = 0, always a hit) is
    // cleared afterwards instead of being tested for in the loop.
    for (int pi0 = wid * NB_PB; pi0 < np; pi0 += (NS_THREADS / 32) * NB_PB) {
        float4 p[NB_PB];
        int found[NB_PB];
#pragma unroll
        for (int b = 0; b < NB_PB; ++b) { p[b] = pos[first + min(pi0 + b, np - 1)]; found[b] = 0; }
        for (int w = 0; w < nwords; ++w) {
            const float4 q = cpos[w * 32 + lane];
            bool in[NB_PB], anyex = false;
#pragma unroll
            for (int b = 0; b < NB_PB; ++b) {
                float dx = p[b].x - q.x, dy = p[b].y - q.y;
                const float dz = p[b].z - q.z;
                if (DEF) { dx = lat.a11 * dx + lat.a12 * dy; dy = lat.a22 * dy; }
                const float d2 = dx * dx + dy * dy + dz * dz;
                in[b] = d2 < rc2;
                anyex = anyex || !(fabsf(d2 - rc2) > band);
            }
            if (__any_sync(0xffffffffu, anyex || !fast)) {       // rare on the screened path: a real branch, not predication
                const int j = __float_as_int(q.w);
                if (j >= 0) {
                    const float4 qe = fast ? pos[j] : q;
#pragma unroll
                    for (int b = 0; b < NB_PB; ++b) {
                        float dx = p[b].x - q.x, dy = p[b].y - q.y;
                        const float dz = p[b].z - q.z;
                        if (DEF) { dx = lat.a11 * dx + lat.a12 * dy; dy = lat.a22 * dy; }
                        const float d2 = dx * dx + dy * dy + dz * dz;
                        if (!fast || !(fabsf(d2 - rc2) > band)) in[b] = dist2(p[b], qe, L, invL, lat) < rc2;
                    }
                }
            }
#pragma unroll
            for (int b = 0; b < NB_PB; ++b) {
                const unsigned m = __ballot_sync(0xffffffffu, in[b]);
                if (lane == 0 && pi0 + b < np) masks[pi0 + b][w] = m;
                found[b] += __popc(m);
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int b = 0; b < NB_PB; ++b)
                if (pi0 + b < np) {
                    const int sc = self0 + pi0 + b;
                    masks[pi0 + b][sc >> 5] &= ~(1u << (sc & 31));
                    cnt[pi0 + b] = found[b] - 1;
                }
        }
    }
    __syncthreads();
    if (tid < 32) {                                           // exclusive prefix of the <= 64 counts, one reservation
        const int c0 = tid < np ? cnt[tid] : 0, c1 = tid + 32 < np ? cnt[tid + 32] : 0;
        int i0 = c0, i1 = c1;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v0 = __shfl_up_sync(0xffffffffu, i0, o), v1 = __shfl_up_sync(0xffffffffu, i1, o);
            if (lane >= o) { i0 += v0; i1 += v1; }
        }
        const int tot0 = __shfl_sync(0xffffffffu, i0, 31), tot1 = __shfl_sync(0xffffffffu, i1, 31);
        loc[tid] = i0 - c0; loc[tid + 32] = tot0 + i1 - c1;
        if (tid == 0) base_s = atomicAdd(cursor, (unsigned long long)(tot0 + tot1));
    }
    __syncthreads();
    const unsigned long long base = base_s;
    for (int pi = wid; pi < np; pi += NS_THREADS / 32) {     // pass B: expand the masks word by word, a lane per candidate
        const int s = first + pi;
        const unsigned long long o = base + (unsigned long long)loc[pi];
        const bool fits = o + (unsigned long long)cnt[pi] <= cap;
        if (lane == 0) { off[s] = fits ? o : 0ull; count[s] = fits ? cnt[pi] : 0; }
        if (!fits) continue;                                  // overflow: empty list here (nothing reads past the array); the
                                                              // host sees cursor > cap later and re-runs with a larger array
        int *dst = idx + o;
        const unsigned lt = (1u << lane) - 1u;
        for (int w = 0; w < nwords; ++w) {                    // ascending candidate order; consecutive hits, consecutive addresses
            const unsigned m = masks[pi][w];
            if ((m >> lane) & 1u) dst[__popc(m & lt)] = __float_as_int(cpos[w * 32 + lane].w);
            dst += __popc(m);
        }
    }
}

__global__ void counts_to_original(const int *count_sorted, const int *order, int N, int *count_orig) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < N) count_orig[order[s]] = count_sorted[s];
}

__global__ void lists_to_original(const int *idx, const unsigned long long *off_sorted, const int *count_sorted, const int *order, int N,
                                  const unsigned long long *off_orig, int *out) {
    int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (s >= N) return;
    unsigned long long lo = off_sorted[s], n = (unsigned long long)count_sorted[s], dst = off_orig[order[s]];
    for (unsigned long long j = lane; j < n; j += 32) out[dst + j] = order[idx[lo + j]];
}

// Heyes-Melrose overlap force (reading R12), 8 lanes per particle over the neighbour list (as the pair kernel), packed output.
__global__ void hs_forces(const float4 *__restrict__ pos, int N, const unsigned long long *__restrict__ off, const int *__restrict__ count,
                          const int *__restrict__ idx, float L, float invL, float two_a, float coef, float *__restrict__ out, const Lat *__restrict__ latp) {
    const Lat lat = *latp;
    const int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 3, gl = threadIdx.x & 7;
    const bool live = s < N;
    const float4 p = live ? pos[s] : make_float4(0.f, 0.f, 0.f, 0.f);
    float fx = 0, fy = 0, fz = 0;
    if (live) {
        for (unsigned long long j = off[s] + gl, hi = off[s] + (unsigned long long)count[s]; j < hi; j += 8) {
            float4 q = pos[idx[j]];
            float dx = min_image(p.x - q.x, L, invL), dy = min_image(p.y - q.y, L, invL), dz = min_image(p.z - q.z, L, invL);
            dx = __fadd_rn(__fmul_rn(lat.a11, dx), __fmul_rn(lat.a12, dy)); dy = __fmul_rn(lat.a22, dy);     // r = A d (exact on the cube)
            float r2 = dx * dx + dy * dy + dz * dz;
            if (r2 < two_a * two_a && r2 > 0.f) {
                float r = sqrtf(r2), g = coef * (two_a - r) / r;
                fx += g * dx; fy += g * dy; fz += g * dz;
            }
        }
    }
    for (int o = 4; o; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
    }
    if (gl == 0 && live) {
        float4 *o4 = reinterpret_cast<float4 *>(out + (size_t)s * 8);
        o4[0] = make_float4(fx, fy, fz, 0.f); o4[1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// Forces of the bond potential U(r) = k |r - r0| of the paper's equilibrium test: a thread per bond,
// positions and output in original numbering, F_i -= k sign(r - r0) rhat_ij, F_j += the same (out is zeroed beforehand).
__global__ void bond_forces(const float4 *__restrict__ posw, const int2 *__restrict__ bonds, int nb, float L, float invL, float k, float r0,
                            float *__restrict__ out, const Lat *__restrict__ latp) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const Lat lat = *latp;
    const int2 ij = bonds[b];
    const float4 p = posw[ij.x], q = posw[ij.y];
    float dx = min_image(p.x - q.x, L, invL), dy = min_image(p.y - q.y, L, invL);
    const float dz = min_image(p.z - q.z, L, invL);
    dx = __fadd_rn(__fmul_rn(lat.a11, dx), __fmul_rn(lat.a12, dy)); dy = __fmul_rn(lat.a22, dy);
    const float r = sqrtf(dx * dx + dy * dy + dz * dz);
    if (!(r > 0.f) || r == r0) return;
    const float g = (r > r0 ? -k : k) / r;
    atomicAdd(out + 3 * (size_t)ij.x, g * dx); atomicAdd(out + 3 * (size_t)ij.x + 1, g * dy); atomicAdd(out + 3 * (size_t)ij.x + 2, g * dz);
    atomicAdd(out + 3 * (size_t)ij.y, -g * dx); atomicAdd(out + 3 * (size_t)ij.y + 1, -g * dy); atomicAdd(out + 3 * (size_t)ij.y + 2, -g * dz);
}

}  // namespace

pse_status pse_bond_forces_orig(pse_ctx *c, float *d_F) {
    ScopedPhase ph(c, PSE_T_REAL);
    CUDA_TRY(c, cudaMemsetAsync(d_F, 0, (size_t)3 * c->N * sizeof(float), c->stream));
    if (c->n_bonds == 0) return PSE_OK;
    bond_forces<<<(c->n_bonds + 127) / 128, 128, 0, c->stream>>>(c->d_posw, c->d_bonds, c->n_bonds, (float)c->L, 1.0f / (float)c->L,
                                                                 (float)c->bond_k, (float)c->bond_r0, d_F, c->d_lat);
    KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_rank_sort(pse_ctx *c, const int *seg_start, int nseg, const int *in, int *out) {
    rank_sort_segments<<<(unsigned)(((size_t)nseg * 32 + 255) / 256), 256, 0, c->stream>>>(seg_start, nseg, in, out); KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_scan_u64(pse_ctx *c, const int *d_in, unsigned long long *d_out, size_t n) { return scan_impl(c, d_in, d_out, n); }
pse_status pse_scan_i32(pse_ctx *c, const int *d_in, int *d_out, size_t n) { return scan_impl(c, d_in, d_out, n); }

pse_status pse_neighbors_impl(pse_ctx *c, const float *d_pos_in) {
    ScopedPhase ph(c, PSE_T_NEIGHBORS);
    const int N = c->N, T = 256, nb = (N + T - 1) / T;
    const float L = (float)c->L, invL = 1.0f / L;
    const Cells nc = c->nc;
    const float3 cell_inv = make_float3((float)(nc.x / c->L), (float)(nc.y / c->L), (float)(nc.z / c->L));
    const float rc = (float)c->rcut, rc2 = rc * rc;
    const Lat *lat = c->d_lat;
    // >> 2 r_c ulp(L): rounding gap between screened and R16 distances (the map by A adds a few more roundings of the same size)
    const float band = 32.f * rc * L * 1.2e-7f;      // the kernel widens it by 4 (|a11| + |a12| + |a22|) on a deformed lattice
    c->have_nbrs = false;
    CUDA_TRY(c, cudaMemsetAsync(c->d_bins, 0, c->bins_n * sizeof(int), c->stream));      // cell and tile counters, one memset
    wrap_and_bin<<<nb, T, 0, c->stream>>>(reinterpret_cast<const float4 *>(d_pos_in), N, L, invL, nc, cell_inv,
                                           c->d_posw, c->d_cell_of, c->d_cell_count, (float)(1.0 / c->h), c->M, c->P, c->nt,
                                           c->d_tile_of, c->d_tile_count, lat); KERNEL_CHECK(c);
    if (c->ncell <= SCAN1_MAX && c->ntile <= SCAN1_MAX) {
        scan_two_ctas<<<2, SCAN1_THREADS, 0, c->stream>>>(c->d_cell_count, c->ncell, c->d_cell_start, c->d_tile_count, c->ntile, c->d_tile_start);
        KERNEL_CHECK(c);
    } else {
        PSE_TRY(pse_scan_i32(c, c->d_cell_count, c->d_cell_start, (size_t)c->ncell));
        PSE_TRY(pse_scan_i32(c, c->d_tile_count, c->d_tile_start, (size_t)c->ntile));
    }
    scatter_to_cells<<<nb, T, 0, c->stream>>>(c->d_cell_of, N, c->d_cell_start, c->d_cell_fill, c->d_order_tmp); KERNEL_CHECK(c);
    pse_rank_sort(c, c->d_cell_start, c->ncell, c->d_order_tmp, c->d_order);
    gather_positions<<<nb, T, 0, c->stream>>>(c->d_posw, c->d_order, N, c->d_pos, c->d_tile_of, c->d_tile_start, c->d_tile_fill, c->d_tile_tmp);
    KERNEL_CHECK(c);
    PSE_TRY(pse_tile_bins(c));
    PSE_TRY(pse_particle_windows(c));
    if (!c->d_nbr_idx) {
        const size_t cap = (size_t)N * 48 + 1024;
        if (cudaMalloc(&c->d_nbr_idx, cap * sizeof(int)) != cudaSuccess) { c->err = "out of memory (neighbour list)"; return PSE_ENOMEM; }
        c->nbr_cap = cap;
    }
    if (!c->nbr_two_pass) {
        // single-pass build into a cursor-allocated index array; {cursor, fallback flag} travel to the pinned mirror behind
        // the kernel and are looked at by pse_neighbors_settle, never here
        CUDA_TRY(c, cudaMemsetAsync(c->d_nbr_ctl, 0, 2 * sizeof(unsigned long long), c->stream));
        if (c->deformed)
            neighbor_build_cell<true><<<c->ncell, NS_THREADS, 0, c->stream>>>(c->d_pos, c->d_cell_start, nc, L, invL, rc2, band, c->d_nbr_count, c->d_nbr_off,
                                                                             c->d_nbr_idx, (unsigned long long)c->nbr_cap, c->d_nbr_ctl,
                                                                             reinterpret_cast<int *>(c->d_nbr_ctl + 1), lat);
        else
            neighbor_build_cell<false><<<c->ncell, NS_THREADS, 0, c->stream>>>(c->d_pos, c->d_cell_start, nc, L, invL, rc2, band, c->d_nbr_count, c->d_nbr_off,
                                                                              c->d_nbr_idx, (unsigned long long)c->nbr_cap, c->d_nbr_ctl,
                                                                              reinterpret_cast<int *>(c->d_nbr_ctl + 1), lat);
        KERNEL_CHECK(c);
        c->nbr_last = c->nbr_slot; c->nbr_slot ^= 1;               // two report slots: pse_step has two builds in flight
        CUDA_TRY(c, cudaMemcpyAsync(c->h_nbr_ctl + 2 * c->nbr_last, c->d_nbr_ctl, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaEventRecord(c->ev_nbr, c->stream));
        c->nbr_pending = true;
    } else {                                                         // general two-pass path (count, scan, fill); synchronises
        neighbor_sweep_cell<false><<<c->ncell, NS_THREADS, 0, c->stream>>>(c->d_pos, c->d_cell_start, nc, L, invL, rc2, c->d_nbr_count,
                                                                            nullptr, nullptr, lat); KERNEL_CHECK(c);
        PSE_TRY(pse_scan_u64(c, c->d_nbr_count, c->d_nbr_off, (size_t)N));
        unsigned long long total = 0;
        CUDA_TRY(c, cudaMemcpyAsync(&total, c->d_nbr_off + N, sizeof(total), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (total > c->nbr_cap) {
            if (c->d_nbr_idx) cudaFree(c->d_nbr_idx);
            c->d_nbr_idx = nullptr; c->nbr_cap = 0;
            size_t cap = (size_t)(total * 1.25) + 1024;
            if (cudaMalloc(&c->d_nbr_idx, cap * sizeof(int)) != cudaSuccess) { c->err = "out of memory (neighbour list)"; return PSE_ENOMEM; }
            c->nbr_cap = cap;
        }
        c->nbr_total = (size_t)total;
        neighbor_sweep_cell<true><<<c->ncell, NS_THREADS, 0, c->stream>>>(c->d_pos, c->d_cell_start, nc, L, invL, rc2, c->d_cell_of,
                                                                           c->d_nbr_off, c->d_nbr_idx, lat); KERNEL_CHECK(c);
        c->nbr_pending = false;
    }
    c->have_nbrs = true;
    return PSE_OK;
}

// Look at what the last single-pass build reported.  *redo = true: the index array was too small (it has been enlarged) or
// a cell exceeded the mask store (the context now takes the two-pass path); the caller must build again and recompute
// whatever consumed the list since (overflowed particles had empty lists, so nothing read out of bounds).  Waits only for
// the build itself; called right after a stream synchronisation it does not wait at all.
pse_status pse_neighbors_settle(pse_ctx *c, bool *redo) {
    *redo = false;
    if (!c->nbr_pending) return PSE_OK;
    CUDA_TRY(c, cudaEventSynchronize(c->ev_nbr));
    c->nbr_pending = false;
    return pse_neighbors_examine(c, c->nbr_last, redo);
}

// the report of one build (slot of h_nbr_ctl), after the stream has passed its read-back
pse_status pse_neighbors_examine(pse_ctx *c, int slot, bool *redo) {
    *redo = false;
    const unsigned long long *ctl = c->h_nbr_ctl + 2 * slot;
    if (ctl[1] != 0) { c->nbr_two_pass = true; c->have_nbrs = false; *redo = true; return PSE_OK; }
    const unsigned long long total = ctl[0];
    if (total > c->nbr_cap) {
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));               // kernels still reading the old array
        cudaFree(c->d_nbr_idx); c->d_nbr_idx = nullptr; c->nbr_cap = 0;
        const size_t cap = (size_t)(total * 1.25) + 1024;
        if (cudaMalloc(&c->d_nbr_idx, cap * sizeof(int)) != cudaSuccess) { c->err = "out of memory (neighbour list)"; return PSE_ENOMEM; }
        c->nbr_cap = cap; c->have_nbrs = false; *redo = true;
        return PSE_OK;
    }
    c->nbr_total = (size_t)total;
    return PSE_OK;
}

// build + settle until the list is complete (the public pse_neighbors and everything outside pse_step)
pse_status pse_neighbors_sync(pse_ctx *c, const float *d_pos) {
    for (int attempt = 0; attempt < 4; ++attempt) {
        bool redo = false;
        PSE_TRY(pse_neighbors_impl(c, d_pos));
        PSE_TRY(pse_neighbors_settle(c, &redo));
        if (!redo) return PSE_OK;
    }
    c->err = "neighbour build did not settle"; return PSE_EOVERFLOW;
}

pse_status pse_get_neighbors_impl(pse_ctx *c, int *d_count, int *d_index, size_t cap, size_t *total) {
    if (!c->have_nbrs) { c->err = "pse_get_neighbors before pse_neighbors"; return PSE_ENOTREADY; }
    const int N = c->N, T = 256;
    if (total) *total = c->nbr_total;
    if (d_count) { counts_to_original<<<(N + T - 1) / T, T, 0, c->stream>>>(c->d_nbr_count, c->d_order, N, d_count); KERNEL_CHECK(c); }
    if (!d_index) return PSE_OK;
    if (cap < c->nbr_total) { c->err = "pse_get_neighbors: index buffer too small"; return PSE_EOVERFLOW; }
    int *cnt = nullptr; unsigned long long *off = nullptr;                    // temporaries released on every path
    pse_status st = PSE_OK;
    if (cudaMalloc(&cnt, (size_t)N * sizeof(int)) != cudaSuccess || cudaMalloc(&off, (size_t)(N + 1) * sizeof(unsigned long long)) != cudaSuccess) {
        c->err = "out of memory (pse_get_neighbors)"; st = PSE_ENOMEM;
    }
    if (st == PSE_OK) { counts_to_original<<<(N + T - 1) / T, T, 0, c->stream>>>(c->d_nbr_count, c->d_order, N, cnt); c->launches++; }
    if (st == PSE_OK) st = pse_scan_u64(c, cnt, off, (size_t)N);
    if (st == PSE_OK) {
        lists_to_original<<<(unsigned)(((size_t)N * 32 + T - 1) / T), T, 0, c->stream>>>(c->d_nbr_idx, c->d_nbr_off, c->d_nbr_count, c->d_order, N, off, d_index);
        c->launches++;
        const cudaError_t e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) { c->err = std::string("pse_get_neighbors: ") + cudaGetErrorString(e); st = PSE_ECUDA; }
    }
    cudaFree(cnt); cudaFree(off);
    return st;
}

pse_status pse_hs_forces_packed(pse_ctx *c, double dt, float *d_out_packed) {
    ScopedPhase ph(c, PSE_T_REAL);
    const int N = c->N, T = 256;
    float coef = (float)(3.0 * M_PI * c->eta * c->a / dt);
    hs_forces<<<(unsigned)(((size_t)N * 8 + T - 1) / T), T, 0, c->stream>>>(c->d_pos, N, c->d_nbr_off, c->d_nbr_count, c->d_nbr_idx, (float)c->L,
                                                                            1.0f / (float)c->L, (float)(2 * c->a), coef, d_out_packed, c->d_lat);
    KERNEL_CHECK(c);
    return PSE_OK;
}

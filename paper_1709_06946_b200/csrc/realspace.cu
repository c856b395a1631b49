// Real-space pair kernel (step a2): [U;E]_alpha = sum_beta M^(r)(x_alpha - x_beta) [F;S]_beta + self term
// (Eqs. 25-27; self terms Eqs. A4/A12), over the neighbour list.
//
// Design: persistent CTAs (2 per SM, 16 warps each or fewer where that fills the last round: pse_real_apply), the table of (F1,F2,Ga,Gb | A,B,D,-) staged once per CTA in shared memory as two
// planar float4 arrays, EIGHT lanes per particle (four particles per warp, four independent idx -> pos -> input chains in
// flight), lanes stride the CSR neighbour list, one 128-bit gather of the neighbour's position and one 256-bit gather of its
// packed input, linear interpolation of the table in r, 7-shuffle reduction of the 8 outputs over the 8 lanes and one
// 32-byte store per particle.  Templated on the component mask of the product.  The paper kept its tables in texture memory
// on a K40; shared memory gives conflict-tolerant 16-byte reads with no L1 pressure on the gathers.
//
// Tensor algebra per pair (rh = unit separation, f = rh.F, t = S rh, q = rh.t):
//   U += F1 (F - rh f) + F2 rh f + Ga t - Gb rh q
//   E += A S + sym(rh (x) w),  w = -Ga F + 2B t + (Gb f + D q) rh     (projected on e1..e5; trace terms drop out)
#include "pse_internal.h"

namespace {

constexpr float RS2 = 0.70710678118654752f;   // 1/sqrt2
constexpr float RS6 = 0.40824829046386302f;   // 1/sqrt6

// MODE = PSE_IN_F | PSE_IN_S | PSE_OUT_U | PSE_OUT_E: terms of absent inputs / outputs are removed at compile time
// (inside GMRES the operator is S -> E: no U accumulation, no F terms, and only the E-part table is read).
// The packed input of a particle ([8] floats, 32-byte aligned = one sector) in ONE 256-bit load (LDG.E.256, new on sm_100)
// instead of two 128-bit ones: a third fewer load instructions and L1 requests per pair.
__device__ __forceinline__ void load_packed8(const float4 *in, int b, float4 &a0, float4 &a1) {
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a0.x), "=f"(a0.y), "=f"(a0.z), "=f"(a0.w), "=f"(a1.x), "=f"(a1.y), "=f"(a1.z), "=f"(a1.w)
                 : "l"(in + 2 * (size_t)b));
}

// DEF: deformed lattice (reading R22): pos holds lattice coordinates, the physical separation is r = A d, three more FMAs per pair.
template <int MODE, bool DEF>
__global__ void __launch_bounds__(512, 2)
real_pairs_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ in, float4 *__restrict__ out, int N,
                  const unsigned long long *__restrict__ off, const int *__restrict__ cnt, const int *__restrict__ idx,
                  const float4 *__restrict__ table, float inv_dr, float L, float invL, const Lat *__restrict__ latp) {
    const Lat lat = DEF ? *latp : Lat{1.f, 0.f, 1.f, 1.f, 0.f, 1.f};   // device memory: a captured step survives pse_set_lattice
    // two planar float4 arrays (U-part functions, E-part functions): a 16-byte row stride spreads random rows over
    // all eight 16-byte bank groups; the interleaved 32-byte rows reached only four (ncu: 17 wavefronts per LDS.128)
    extern __shared__ float4 tab[];               // tabU[PSE_NTAB] then tabE[PSE_NTAB]
    float4 *tabU = tab, *tabE = tab + PSE_NTAB;
    constexpr bool INF = MODE & PSE_IN_F, INS = MODE & PSE_IN_S, OUTU = MODE & PSE_OUT_U, OUTE = MODE & PSE_OUT_E;
    constexpr bool NEED_TU = (OUTU) || (INF && OUTE), NEED_TE = INS && OUTE;
    // only the half of the table the component mask reads is staged (32 KB per CTA less for S -> E); row 0 of both halves
    // is always there for the self term
    for (int i = threadIdx.x; i < PSE_NTAB; i += blockDim.x) {
        if (NEED_TU || i == 0) tabU[i] = table[2 * i];
        if (NEED_TE || i == 0) tabE[i] = table[2 * i + 1];
    }
    __syncthreads();
    // G = 8 lanes per particle (4 particles per warp): a list of ~51 entries fills 7 passes of 8 lanes to 91 %, two passes
    // of 32 lanes only to 80 % (measured, config 3 / config 4, us per launch: 32 lanes 44.9 / 719, 16: 40.3 / 608, 8: 41.0 / 585)
    constexpr int G = 8, PPW = 32 / G;
    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5, gl = lane & (G - 1), grp = lane / G;
    for (int ws = blockIdx.x * wpb + (threadIdx.x >> 5); ws * PPW < N; ws += gridDim.x * wpb) {
        const int s = ws * PPW + grp;
        const bool live = s < N;
        const float4 p = live ? pos[s] : make_float4(0.f, 0.f, 0.f, 0.f);
        float u0 = 0, u1 = 0, u2 = 0, e0 = 0, e1 = 0, e2 = 0, e3 = 0, e4 = 0;
        const unsigned long long lo = live ? off[s] : 0ull, hi = lo + (unsigned long long)(live ? cnt[s] : 0);
        // software pipeline of depth one on the dependent chain idx -> pos: the next neighbour's index and position
        // are requested while the current pair is evaluated (ncu: 42 % of the stall samples sat on these two waits)
        unsigned long long j = lo + gl;
        int b = j < hi ? idx[j] : 0;
        float4 q4 = pos[b];
        for (; j < hi; j += G) {
            float4 a0, a1;
            if (INS) load_packed8(in, b, a0, a1);
            else { a0 = in[2 * b]; a0.w = 0.f; a1 = make_float4(0.f, 0.f, 0.f, 0.f); }
            if (!INF) { a0.x = 0.f; a0.y = 0.f; a0.z = 0.f; }
            const int bn = (j + G < hi) ? idx[j + G] : b;
            float dx = p.x - q4.x, dy = p.y - q4.y, dz = p.z - q4.z;
            dx -= L * rintf(dx * invL); dy -= L * rintf(dy * invL); dz -= L * rintf(dz * invL);
            if (DEF) { dx = lat.a11 * dx + lat.a12 * dy; dy = lat.a22 * dy; }
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float rinv = rsqrtf(fmaxf(r2, 1e-30f)), r = r2 * rinv;
            const float rx = dx * rinv, ry = dy * rinv, rz = dz * rinv;
            float tt = r * inv_dr;
            int it = min((int)tt, PSE_NTAB - 2);
            const float w1 = tt - (float)it, w0 = 1.f - w1;
            const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
            const float4 ta = NEED_TU ? tabU[it] : zero4, tc = NEED_TU ? tabU[it + 1] : zero4;
            const float4 tb = NEED_TE ? tabE[it] : zero4, td = NEED_TE ? tabE[it + 1] : zero4;
            const float F1 = w0 * ta.x + w1 * tc.x, F2 = w0 * ta.y + w1 * tc.y, Ga = w0 * ta.z + w1 * tc.z, Gb = w0 * ta.w + w1 * tc.w;
            const float A = w0 * tb.x + w1 * td.x, B = w0 * tb.y + w1 * td.y, D = w0 * tb.z + w1 * td.z;
            const float4 qn = pos[bn];
            // S_beta from its 5 coordinates
            const float sxx = a0.w * RS2 - a1.x * RS6, syy = -a0.w * RS2 - a1.x * RS6, szz = 2.f * a1.x * RS6;
            const float sxy = a1.y * RS2, sxz = a1.z * RS2, syz = a1.w * RS2;
            const float f = rx * a0.x + ry * a0.y + rz * a0.z;
            const float tx = sxx * rx + sxy * ry + sxz * rz, ty = sxy * rx + syy * ry + syz * rz, tz = sxz * rx + syz * ry + szz * rz;
            const float q = rx * tx + ry * ty + rz * tz;
            const float cu = (F2 - F1) * f - Gb * q;
            if (OUTU) {
                u0 += F1 * a0.x + cu * rx + Ga * tx;
                u1 += F1 * a0.y + cu * ry + Ga * ty;
                u2 += F1 * a0.z + cu * rz + Ga * tz;
            }
            const float cw = Gb * f + D * q, B2 = 2.f * B;
            const float wx = -Ga * a0.x + B2 * tx + cw * rx, wy = -Ga * a0.y + B2 * ty + cw * ry, wz = -Ga * a0.z + B2 * tz + cw * rz;
            const float pxx = rx * wx, pyy = ry * wy, pzz = rz * wz;
            if (OUTE) {
                e0 += A * a0.w + (pxx - pyy) * RS2;
                e1 += A * a1.x + (2.f * pzz - pxx - pyy) * RS6;
                e2 += A * a1.y + (rx * wy + ry * wx) * RS2;
                e3 += A * a1.z + (rx * wz + rz * wx) * RS2;
                e4 += A * a1.w + (ry * wz + rz * wy) * RS2;
            }
            b = bn;
            q4 = qn;
        }
        // self term (r -> 0 limit: F1(0) F and A(0) S) added by the group's first lane before the reduction
        if (gl == 0 && live) {
            const float4 a0 = in[2 * s], a1 = in[2 * s + 1], t0 = tabU[0], t1 = tabE[0];
            if (INF && OUTU) { u0 += t0.x * a0.x; u1 += t0.x * a0.y; u2 += t0.x * a0.z; }
            if (INS && OUTE) { e0 += t1.x * a0.w; e1 += t1.x * a1.x; e2 += t1.x * a1.y; e3 += t1.x * a1.z; e4 += t1.x * a1.w; }
        }
        const float part[8] = {u0, u1, u2, e0, e1, e2, e3, e4};
        // 8 sums over 8 lanes in 4 + 2 + 1 shuffles: every step halves the values a lane carries; lane gl ends with component gl
        const bool h1 = gl & 4, h2 = gl & 2, h3 = gl & 1;
        float r4[4], r2[2];
#pragma unroll
        for (int c = 0; c < 4; ++c) r4[c] = (h1 ? part[c + 4] : part[c]) + __shfl_xor_sync(0xffffffffu, h1 ? part[c] : part[c + 4], 4);
#pragma unroll
        for (int c = 0; c < 2; ++c) r2[c] = (h2 ? r4[c + 2] : r4[c]) + __shfl_xor_sync(0xffffffffu, h2 ? r4[c] : r4[c + 2], 2);
        const float r = (h3 ? r2[1] : r2[0]) + __shfl_xor_sync(0xffffffffu, h3 ? r2[0] : r2[1], 1);
        if (live) reinterpret_cast<float *>(out)[(size_t)s * 8 + gl] = r;
    }
}

}  // namespace

constexpr size_t REAL_SMEM = (size_t)PSE_NTAB * 2 * sizeof(float4);

template <int MODE>
static pse_status launch_real(pse_ctx *c, const float *d_in, float *d_out, int grid, int threads) {
    const float4 *in4 = reinterpret_cast<const float4 *>(d_in), *tab = reinterpret_cast<const float4 *>(c->d_table);
    float4 *out4 = reinterpret_cast<float4 *>(d_out);
    const float inv_dr = (float)(1.0 / c->tab_dr), L = (float)c->L, invL = 1.0f / (float)c->L;
    if (c->deformed)
        real_pairs_kernel<MODE, true><<<grid, threads, REAL_SMEM, c->stream>>>(c->d_pos, in4, out4, c->N, c->d_nbr_off, c->d_nbr_count, c->d_nbr_idx, tab,
                                                                         inv_dr, L, invL, c->d_lat);
    else
        real_pairs_kernel<MODE, false><<<grid, threads, REAL_SMEM, c->stream>>>(c->d_pos, in4, out4, c->N, c->d_nbr_off, c->d_nbr_count, c->d_nbr_idx, tab,
                                                                          inv_dr, L, invL, c->d_lat);
    KERNEL_CHECK(c);
    return PSE_OK;
}

// dynamic shared-memory opt-in of every instantiation on the context's device (called by pse_create)
pse_status pse_real_init(pse_ctx *c) {
#define PSE_REAL_ATTR(M) CUDA_TRY(c, cudaFuncSetAttribute(real_pairs_kernel<M, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)REAL_SMEM)); \
                         CUDA_TRY(c, cudaFuncSetAttribute(real_pairs_kernel<M, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)REAL_SMEM))
    PSE_REAL_ATTR(PSE_IN_S | PSE_OUT_E); PSE_REAL_ATTR(PSE_IN_F | PSE_OUT_E); PSE_REAL_ATTR(PSE_IN_F | PSE_IN_S | PSE_OUT_U);
    PSE_REAL_ATTR(PSE_IN_S | PSE_OUT_U); PSE_REAL_ATTR(PSE_IN_F | PSE_OUT_U); PSE_REAL_ATTR(PSE_MODE_ALL);
#undef PSE_REAL_ATTR
    return PSE_OK;
}

pse_status pse_real_apply(pse_ctx *c, const float *d_in, float *d_out, int mode) {
    ScopedPhase ph(c, PSE_T_REAL);
    int grid = 2 * c->nsm, wpb = 512 / 32;
    const long long tasks = ((long long)c->N + 3) / 4;           // one warp pass = 4 particles
    if ((long long)grid * wpb >= tasks) grid = (int)((tasks + wpb - 1) / wpb);
    else {
        // The persistent warps take whole tasks round-robin, so a launch lasts ceil(tasks / warps) rounds and the last one may be
        // nearly empty (config 3: 3.46 rounds of 16-warp CTAs).  Measured (S -> E against N at config 3's density, 12 to 16 warps):
        // time = 7.3 us + 0.44 us x cost, where a full round costs the number of warps that share an SM's L1 and a last round filled
        // to a fraction f costs about min(1, 0.45 + 1.2 f) of a full one (its dependent loads are paid whatever f is).  Narrower
        // CTAs whose last round is full win where that model says so by 5 %: 14 warps at config 3 (3.95 rounds), 33.5 -> 31.3 us
        // per launch; a launch barely over one round (N = 20 000) and large N keep 16 warps.
        auto cost = [&](int w) {
            const double R = (double)tasks / ((double)grid * w), full = std::floor(R), f = R - full;
            return w * (full + (f > 0 ? std::min(1.0, 0.45 + 1.2 * f) : 0.0));
        };
        double best = 0.95 * cost(16);
        for (int w = 15; w >= 12; --w)
            if (cost(w) < best) { best = cost(w); wpb = w; }
    }
    const int threads = wpb * 32;
    // unrequested outputs are written as zeros; absent inputs must be zero in d_in (they are skipped, not read as data)
    switch (mode) {
        case PSE_IN_S | PSE_OUT_E: return launch_real<PSE_IN_S | PSE_OUT_E>(c, d_in, d_out, grid, threads);
        case PSE_IN_F | PSE_OUT_E: return launch_real<PSE_IN_F | PSE_OUT_E>(c, d_in, d_out, grid, threads);
        case PSE_IN_F | PSE_IN_S | PSE_OUT_U: return launch_real<PSE_IN_F | PSE_IN_S | PSE_OUT_U>(c, d_in, d_out, grid, threads);
        case PSE_IN_S | PSE_OUT_U: return launch_real<PSE_IN_S | PSE_OUT_U>(c, d_in, d_out, grid, threads);
        case PSE_IN_F | PSE_OUT_U: return launch_real<PSE_IN_F | PSE_OUT_U>(c, d_in, d_out, grid, threads);
        default: return launch_real<PSE_MODE_ALL>(c, d_in, d_out, grid, threads);
    }
}

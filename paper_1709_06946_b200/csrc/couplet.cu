// Full couplet: [U; Omega; E] = M [F; L; S], Eq. (31) with the decomposition of Eqs. (32)-(35)
// (PAPER.md:175-185).  The force / stresslet block is the tuned 8-component path; this file adds the torque and
// angular-velocity rows around it without touching it (reading R21 fixes the conventions by the physics:
// a torque acts on the fluid as (1/2) curl(L delta), the angular velocity is the sphere average of (1/2) curl u, both
// with the couplet shape factor s1 = 3 j1(ka)/ka of PAPER.md:111):
//
//   wave space   fh = s0 Fh + (i/2) s1 k x Lh - i s1 Sh.k ;  uh = B (I - kh kh) fh ;
//                Uh = s0 uh ;  Omega_h = (i/2) s1 k x uh ;  Eh^q = i s1 (e^q k).uh
//                -> the torque is spread on 3 planes of its own and transformed into c->d_spec_rot, ONE scaling kernel reads the
//                   11 spectra and writes 11, the three Omega planes come back through the same 3-plane transform and interpolation.
//   real space   U     += T' L x rh
//                Omega += T' F x rh + Y0 L + Y2 (rh rh.L - L/3) + 2 Y2 (S rh) x rh
//                E     += 2 Y2 sym[ rh (x) (rh x L) ]
//                with (T', Y0, Y2) = (T/2, Z0/6, Z2/4)/(6 pi eta a), T = G1 - G2 (the antisymmetric part of Eq. 26), from a
//                table of their own at the nodes of the main table (tables.cu), in real_pairs_full_kernel: the 11-component pair
//                sum in one sweep, eight lanes per particle as in the 8-component pair kernel.
#include <algorithm>
#include <cmath>
#include "pse_internal.h"
#include "wave_scale.cuh"

namespace {

constexpr float RS2 = 0.70710678118654752f, RS6 = 0.40824829046386302f;

// The 11-component pair sum in ONE sweep over the neighbour list: the tensor algebra of real_pairs_kernel (realspace.cu) plus the
// rotational terms of the file header on one set of gathers, with both tables in shared memory (64 + 32 KB).  Eight lanes per
// particle, 384 threads, two CTAs per SM (72 registers: 11 accumulators, 11 inputs).  (A second sweep that added the rotational
// terms to the 8-component kernel's result cost 48 us on top of its 37 us at config 3; this one takes 60 us.)
constexpr size_t FULL_SMEM = (size_t)PSE_NTAB * 3 * sizeof(float4);

__global__ void __launch_bounds__(384, 2)
real_pairs_full_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ in8, const float4 *__restrict__ inL, float *__restrict__ out8,
                       float *__restrict__ outW, int N, const unsigned long long *__restrict__ off, const int *__restrict__ cnt,
                       const int *__restrict__ idx, const float4 *__restrict__ table, const float4 *__restrict__ rtable, float inv_dr, float L,
                       float invL, const Lat *__restrict__ latp) {
    const Lat lat = *latp;
    extern __shared__ float4 ftab[];                           // tabU[NTAB] | tabE[NTAB] | tabR[NTAB]
    float4 *tabU = ftab, *tabE = ftab + PSE_NTAB, *tabR = ftab + 2 * PSE_NTAB;
    for (int i = threadIdx.x; i < PSE_NTAB; i += blockDim.x) { tabU[i] = table[2 * i]; tabE[i] = table[2 * i + 1]; tabR[i] = rtable[i]; }
    __syncthreads();
    const int gl = threadIdx.x & 7, grp = (threadIdx.x & 31) >> 3, wpb = blockDim.x >> 5;
    for (int ws = blockIdx.x * wpb + (threadIdx.x >> 5); ws * 4 < N; ws += gridDim.x * wpb) {
        const int s = ws * 4 + grp;
        const bool live = s < N;
        const float4 p = live ? pos[s] : make_float4(0.f, 0.f, 0.f, 0.f);
        float acc[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};          // U (3), E (5), Omega (3)
        const unsigned long long lo = live ? off[s] : 0ull, hi = lo + (unsigned long long)(live ? cnt[s] : 0);
        unsigned long long j = lo + gl;
        int b = j < hi ? idx[j] : 0;
        float4 q4 = pos[b];
        for (; j < hi; j += 8) {
            const float4 a0 = in8[2 * b], a1 = in8[2 * b + 1], l4 = inL[2 * b];
            const int bn = (j + 8 < hi) ? idx[j + 8] : b;
            float dx = p.x - q4.x, dy = p.y - q4.y, dz = p.z - q4.z;
            dx -= L * rintf(dx * invL); dy -= L * rintf(dy * invL); dz -= L * rintf(dz * invL);
            dx = lat.a11 * dx + lat.a12 * dy; dy = lat.a22 * dy;
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float rinv = rsqrtf(fmaxf(r2, 1e-30f)), r = r2 * rinv;
            const float rx = dx * rinv, ry = dy * rinv, rz = dz * rinv;
            const float tt = r * inv_dr;
            const int it = min((int)tt, PSE_NTAB - 2);
            const float w1 = tt - (float)it, w0 = 1.f - w1;
            const float4 ta = tabU[it], tc = tabU[it + 1], tb = tabE[it], td = tabE[it + 1], ra = tabR[it], rb = tabR[it + 1];
            const float F1 = w0 * ta.x + w1 * tc.x, F2 = w0 * ta.y + w1 * tc.y, Ga = w0 * ta.z + w1 * tc.z, Gb = w0 * ta.w + w1 * tc.w;
            const float A = w0 * tb.x + w1 * td.x, B = w0 * tb.y + w1 * td.y, D = w0 * tb.z + w1 * td.z;
            const float Tq = w0 * ra.x + w1 * rb.x, Y0 = w0 * ra.y + w1 * rb.y, Y2 = w0 * ra.z + w1 * rb.z;
            const float4 qn = pos[bn];
            const float sxx = a0.w * RS2 - a1.x * RS6, syy = -a0.w * RS2 - a1.x * RS6, szz = 2.f * a1.x * RS6;
            const float sxy = a1.y * RS2, sxz = a1.z * RS2, syz = a1.w * RS2;
            const float f = rx * a0.x + ry * a0.y + rz * a0.z;
            const float tx = sxx * rx + sxy * ry + sxz * rz, ty = sxy * rx + syy * ry + syz * rz, tz = sxz * rx + syz * ry + szz * rz;
            const float q = rx * tx + ry * ty + rz * tz;
            const float cx = l4.y * rz - l4.z * ry, cy = l4.z * rx - l4.x * rz, cz = l4.x * ry - l4.y * rx;      // L x rh
            const float gx = a0.y * rz - a0.z * ry, gy = a0.z * rx - a0.x * rz, gz = a0.x * ry - a0.y * rx;      // F x rh
            const float cu = (F2 - F1) * f - Gb * q;
            acc[0] += F1 * a0.x + cu * rx + Ga * tx + Tq * cx;
            acc[1] += F1 * a0.y + cu * ry + Ga * ty + Tq * cy;
            acc[2] += F1 * a0.z + cu * rz + Ga * tz + Tq * cz;
            const float cw = Gb * f + D * q, B2 = 2.f * B, Y22 = 2.f * Y2;
            // E += A S + sym[rh (x) w],  w = -Ga F + 2B t + (Gb f + D q) rh + 2 Y2 (rh x L)
            const float wx = -Ga * a0.x + B2 * tx + cw * rx - Y22 * cx, wy = -Ga * a0.y + B2 * ty + cw * ry - Y22 * cy,
                        wz = -Ga * a0.z + B2 * tz + cw * rz - Y22 * cz;
            const float pxx = rx * wx, pyy = ry * wy, pzz = rz * wz;
            acc[3] += A * a0.w + (pxx - pyy) * RS2;
            acc[4] += A * a1.x + (2.f * pzz - pxx - pyy) * RS6;
            acc[5] += A * a1.y + (rx * wy + ry * wx) * RS2;
            acc[6] += A * a1.z + (rx * wz + rz * wx) * RS2;
            acc[7] += A * a1.w + (ry * wz + rz * wy) * RS2;
            const float rl = rx * l4.x + ry * l4.y + rz * l4.z, third = 1.f / 3.f;
            acc[8] += Tq * gx + Y0 * l4.x + Y2 * (rx * rl - third * l4.x) + Y22 * (ty * rz - tz * ry);
            acc[9] += Tq * gy + Y0 * l4.y + Y2 * (ry * rl - third * l4.y) + Y22 * (tz * rx - tx * rz);
            acc[10] += Tq * gz + Y0 * l4.z + Y2 * (rz * rl - third * l4.z) + Y22 * (tx * ry - ty * rx);
            b = bn; q4 = qn;
        }
        if (gl == 0 && live) {                                       // self terms F1(0) F, A(0) S, Z0(0)/6 L
            const float4 a0 = in8[2 * s], a1 = in8[2 * s + 1], l4 = inL[2 * s];
            const float f1 = tabU[0].x, a_ = tabE[0].x, y0 = tabR[0].y;
            acc[0] += f1 * a0.x; acc[1] += f1 * a0.y; acc[2] += f1 * a0.z;
            acc[3] += a_ * a0.w; acc[4] += a_ * a1.x; acc[5] += a_ * a1.y; acc[6] += a_ * a1.z; acc[7] += a_ * a1.w;
            acc[8] += y0 * l4.x; acc[9] += y0 * l4.y; acc[10] += y0 * l4.z;
        }
#pragma unroll
        for (int c = 0; c < 11; ++c)
            for (int o = 4; o; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
        if (live) {
            float mine = acc[0], w = acc[8];
#pragma unroll
            for (int c = 1; c < 8; ++c) mine = gl == c ? acc[c] : mine;
            w = gl == 1 ? acc[9] : (gl == 2 ? acc[10] : w);
            out8[(size_t)s * 8 + gl] = mine;
            outW[(size_t)s * 8 + gl] = gl < 3 ? w : 0.f;
        }
    }
}

// a5 for the full couplet: the 8 spectra of (F, S) in `spec`, the 3 of L in `rot`; all 11 are overwritten with (U, E) and Omega
__global__ void __launch_bounds__(256) scale_full_kernel(cufftComplex *spec, cufftComplex *rot, ScaleParams sp) {
    const unsigned plane = (unsigned)sp.M * (unsigned)sp.Mh, rem = blockIdx.x * blockDim.x + threadIdx.x;
    if (rem >= plane) return;
    const int ix = (int)blockIdx.y, iy = (int)(rem / (unsigned)sp.Mh), iz = (int)(rem - (unsigned)iy * (unsigned)sp.Mh);
    const size_t nmode = (size_t)plane * sp.M, o = (size_t)ix * plane + rem;
    const float2 zero = make_float2(0.f, 0.f);
    float kx, ky, kz;
    if (!mode_k(sp, ix, iy, iz, kx, ky, kz)) {
#pragma unroll
        for (int c = 0; c < 8; ++c) spec[c * nmode + o] = zero;
#pragma unroll
        for (int c = 0; c < 3; ++c) rot[c * nmode + o] = zero;
        return;
    }
    const float k2 = kx * kx + ky * ky + kz * kz, kn = sqrtf(k2), ka = kn * sp.a;
    float s0, s1;
    shape_factors(ka, s0, s1);
    const float q = k2 * sp.inv4xi2;
    const float dw = __ldg(sp.dec + ix) * __ldg(sp.dec + iy) * __ldg(sp.dec + iz);
    const float Bt = sp.c_mv * sp.inv_eta * (1.f + q) * __expf(-q) / k2 * dw * dw;
    float2 F[3], S[5], Lh[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { F[c] = spec[c * nmode + o]; Lh[c] = rot[c * nmode + o]; }
#pragma unroll
    for (int c = 0; c < 5; ++c) S[c] = spec[(3 + c) * nmode + o];
    float2 sk[3], kl[3];                                             // S.k and k x L, real and imaginary parts
#pragma unroll
    for (int ri = 0; ri < 2; ++ri) {
        const float s1c = ri ? S[0].y : S[0].x, s2c = ri ? S[1].y : S[1].x, s3c = ri ? S[2].y : S[2].x, s4c = ri ? S[3].y : S[3].x,
                    s5c = ri ? S[4].y : S[4].x;
        const float sxx = s1c * WS_RS2 - s2c * WS_RS6, syy = -s1c * WS_RS2 - s2c * WS_RS6, szz = 2.f * s2c * WS_RS6;
        const float sxy = s3c * WS_RS2, sxz = s4c * WS_RS2, syz = s5c * WS_RS2;
        const float vx = sxx * kx + sxy * ky + sxz * kz, vy = sxy * kx + syy * ky + syz * kz, vz = sxz * kx + syz * ky + szz * kz;
        const float lx = ri ? Lh[0].y : Lh[0].x, ly = ri ? Lh[1].y : Lh[1].x, lz = ri ? Lh[2].y : Lh[2].x;
        const float cx = ky * lz - kz * ly, cy = kz * lx - kx * lz, cz = kx * ly - ky * lx;
        if (ri) { sk[0].y = vx; sk[1].y = vy; sk[2].y = vz; kl[0].y = cx; kl[1].y = cy; kl[2].y = cz; }
        else { sk[0].x = vx; sk[1].x = vy; sk[2].x = vz; kl[0].x = cx; kl[1].x = cy; kl[2].x = cz; }
    }
    // fh = s0 F - i s1 sk + (i/2) s1 kl :   -i z = (z.im, -z.re),  i z = (-z.im, z.re)
    const float h1 = 0.5f * s1;
    float2 f[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) f[c] = make_float2(s0 * F[c].x + s1 * sk[c].y - h1 * kl[c].y, s0 * F[c].y - s1 * sk[c].x + h1 * kl[c].x);
    const float ik2 = 1.f / k2;
    const float2 kf = make_float2((kx * f[0].x + ky * f[1].x + kz * f[2].x) * ik2, (kx * f[0].y + ky * f[1].y + kz * f[2].y) * ik2);
    const float2 ux = make_float2(Bt * (f[0].x - kx * kf.x), Bt * (f[0].y - kx * kf.y));
    const float2 uy = make_float2(Bt * (f[1].x - ky * kf.x), Bt * (f[1].y - ky * kf.y));
    const float2 uz = make_float2(Bt * (f[2].x - kz * kf.x), Bt * (f[2].y - kz * kf.y));
    write_outputs(spec, nmode, o, s0, s1, kx, ky, kz, ux, uy, uz, PSE_OUT_U | PSE_OUT_E);
    // Omega_h = (i/2) s1 k x uh
    const float2 wx = make_float2(ky * uz.x - kz * uy.x, ky * uz.y - kz * uy.y);
    const float2 wy = make_float2(kz * ux.x - kx * uz.x, kz * ux.y - kx * uz.y);
    const float2 wz = make_float2(kx * uy.x - ky * ux.x, kx * uy.y - ky * ux.y);
    rot[o] = make_float2(-h1 * wx.y, h1 * wx.x);
    rot[nmode + o] = make_float2(-h1 * wy.y, h1 * wy.x);
    rot[2 * nmode + o] = make_float2(-h1 * wz.y, h1 * wz.x);
}

// in8 = (F of a | S of b): the force slots of one packed vector, the stresslet slots of another (a may be NULL = 0)
__global__ void k_merge_force_stresslet(const float4 *a, const float4 *b, int N, float4 *out) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const float4 f = a ? a[2 * s] : make_float4(0.f, 0.f, 0.f, 0.f), b0 = b[2 * s];
    out[2 * s] = make_float4(f.x, f.y, f.z, b0.w);
    out[2 * s + 1] = b[2 * s + 1];
}

// noise [N][11] = (Ux,Uy,Uz, Ox,Oy,Oz, e1..e5) per particle, original numbering -> wide packed vector [2][N][8], sorted numbering
__global__ void k_pack11(const float *v11, const int *order, int N, float4 *wide) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const float *v = v11 + 11 * (size_t)order[s];
    wide[2 * s] = make_float4(v[0], v[1], v[2], v[6]);
    wide[2 * s + 1] = make_float4(v[7], v[8], v[9], v[10]);
    wide[2 * (size_t)N + 2 * s] = make_float4(v[3], v[4], v[5], 0.f);
    wide[2 * (size_t)N + 2 * s + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// x_out = x_in + dt U (original numbering), wrapped into [0, L) per component on the cube only (on a deformed lattice that is not
// a lattice translation; pse_neighbors takes any image)
__global__ void k_advance_full(const float4 *pos_in, const float *U, float dt, float L, float invL, int N, float4 *pos_out, int wrap) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float4 p = pos_in[i];
    p.x += dt * U[3 * i]; p.y += dt * U[3 * i + 1]; p.z += dt * U[3 * i + 2];
    if (wrap) {
        p.x -= L * floorf(p.x * invL); p.y -= L * floorf(p.y * invL); p.z -= L * floorf(p.z * invL);
        if (p.x >= L || p.x < 0.f) p.x = 0.f;
        if (p.y >= L || p.y < 0.f) p.y = 0.f;
        if (p.z >= L || p.z < 0.f) p.z = 0.f;
    }
    pos_out[i] = p;
}

}  // namespace

void pse_couplet_free(pse_ctx *c) {
    cudaFree(c->d_rot_table); cudaFree(c->d_spec_rot); cudaFree(c->d_rot_in); cudaFree(c->d_rot_out); cudaFree(c->d_rot_tmp);
    cudaFree(c->d_rot_w); cudaFree(c->d_rot_y); cudaFree(c->d_rot_u);
    c->d_rot_table = nullptr; c->d_spec_rot = nullptr; c->d_rot_in = c->d_rot_out = c->d_rot_tmp = nullptr;
    c->d_rot_w = c->d_rot_y = c->d_rot_u = nullptr;
}

// table, spectrum and packed vectors of the torque rows: made by the first call that needs them (synchronises once)
static pse_status ensure_couplet(pse_ctx *c) {
    if (c->d_rot_table) return PSE_OK;
    std::vector<float> tab;
    pse_build_rot_table(c->a, c->eta, c->xi, c->rcut, PSE_NTAB, tab);
    const size_t nmode = (size_t)c->M * c->M * c->Mh, vec = (size_t)c->N * 8 * sizeof(float);
    if (cudaMalloc(&c->d_spec_rot, 3 * nmode * sizeof(cufftComplex)) != cudaSuccess || cudaMalloc(&c->d_rot_in, vec) != cudaSuccess ||
        cudaMalloc(&c->d_rot_out, vec) != cudaSuccess || cudaMalloc(&c->d_rot_tmp, vec) != cudaSuccess ||
        cudaMalloc(&c->d_rot_w, 2 * vec) != cudaSuccess || cudaMalloc(&c->d_rot_y, 2 * vec) != cudaSuccess || cudaMalloc(&c->d_rot_u, 2 * vec) != cudaSuccess ||
        cudaMalloc(&c->d_rot_table, tab.size() * sizeof(float)) != cudaSuccess) {
        cudaGetLastError();
        pse_couplet_free(c);
        c->err = "out of memory (full-couplet buffers)"; return PSE_ENOMEM;
    }
    CUDA_TRY(c, cudaMemcpy(c->d_rot_table, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice));
    CUDA_TRY(c, cudaFuncSetAttribute(real_pairs_full_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FULL_SMEM));
    return PSE_OK;
}

// out8 (U, E) and outW (Omega in slots 0-2) = M [in8 (F, S); inL (L in slots 0-2)], packed vectors in sorted numbering
static pse_status apply_full_packed(pse_ctx *c, const float *in8, const float *inL, float *out8, float *outW, int which) {
    const size_t vec = (size_t)c->N * 8 * sizeof(float);
    if (which & PSE_REAL) {
        ScopedPhase ph(c, PSE_T_REAL);
        const int wpb = 384 / 32;
        int grid = 2 * c->nsm;
        if ((long long)grid * wpb * 4 > c->N) grid = (c->N + wpb * 4 - 1) / (wpb * 4);
        real_pairs_full_kernel<<<grid, 384, FULL_SMEM, c->stream>>>(c->d_pos, reinterpret_cast<const float4 *>(in8), reinterpret_cast<const float4 *>(inL),
                                                                    out8, outW, c->N, c->d_nbr_off, c->d_nbr_count, c->d_nbr_idx,
                                                                    reinterpret_cast<const float4 *>(c->d_table), reinterpret_cast<const float4 *>(c->d_rot_table),
                                                                    (float)(1.0 / c->tab_dr), (float)c->L, 1.0f / (float)c->L, c->d_lat);
        KERNEL_CHECK(c);
    } else {
        CUDA_TRY(c, cudaMemsetAsync(out8, 0, vec, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(outW, 0, vec, c->stream));
    }
    if (!(which & PSE_WAVE)) return PSE_OK;
    // torque planes first (they pass through planes 0-2 of the grid array), then the eight planes of (F, S)
    PSE_TRY(pse_wave_spread(c, inL, 1));
    { ScopedPhase ph(c, PSE_T_FFT_FWD); CUFFT_TRY(c, cufftExecR2C(c->plan_r2c[1], c->d_grid, c->d_spec_rot)); c->launches++; }
    PSE_TRY(pse_wave_spread(c, in8, 0));
    { ScopedPhase ph(c, PSE_T_FFT_FWD); CUFFT_TRY(c, cufftExecR2C(c->plan_r2c[0], c->d_grid, c->d_spec)); c->launches++; }
    {
        ScopedPhase ph(c, PSE_T_SCALE);
        scale_full_kernel<<<dim3((unsigned)((c->M * c->Mh + 255) / 256), (unsigned)c->M), 256, 0, c->stream>>>(c->d_spec, c->d_spec_rot, make_scale_params(c));
        KERNEL_CHECK(c);
    }
    { ScopedPhase ph(c, PSE_T_FFT_INV); CUFFT_TRY(c, cufftExecC2R(c->plan_c2r[0], c->d_spec, c->d_grid)); c->launches++; }
    PSE_TRY(pse_wave_interp(c, out8, true, 3));
    { ScopedPhase ph(c, PSE_T_FFT_INV); CUFFT_TRY(c, cufftExecC2R(c->plan_c2r[1], c->d_spec_rot, c->d_grid)); c->launches++; }
    return pse_wave_interp(c, outW, true, 1);
}

// the real-space half on a wide vector [2][N][8]: (U, E | Omega) = M_r (F, S | L)
static pse_status real_full_wide(pse_ctx *c, const float *d_in, float *d_out) {
    const size_t half = (size_t)c->N * 8;
    return apply_full_packed(c, d_in, d_in + half, d_out, d_out + half, PSE_REAL);
}

extern "C" {

pse_status pse_brownian_full(pse_ctx *c, double dt, const float *d_noise_real, const float *d_noise_wave, float *d_UB, float *d_WB, float *d_EB,
                             int *lanczos_iters) {
    if (!c || !(dt > 0) || !d_noise_real || !d_noise_wave) return PSE_EINVAL;
    if (!c->have_nbrs) { c->err = "pse_brownian_full before pse_neighbors"; return PSE_ENOTREADY; }
    PSE_TRY(ensure_couplet(c));
    const size_t half = (size_t)c->N * 8;
    k_pack11<<<(c->N + 255) / 256, 256, 0, c->stream>>>(d_noise_real, c->d_order, c->N, reinterpret_cast<float4 *>(c->d_rot_w)); KERNEL_CHECK(c);
    pse_status st = pse_lanczos_sqrt_wide(c, c->d_rot_w, c->d_rot_y, lanczos_iters, 2, real_full_wide, c->d_rot_u);
    if (st != PSE_OK && st != PSE_ENOCONV) return st;
    PSE_TRY(pse_wave_brownian(c, d_noise_wave, c->d_rot_y, true, c->d_rot_y + half));
    const float amp = (float)std::sqrt(2.0 * c->kT / dt);
    if (d_UB || d_EB) PSE_TRY(pse_unpack(c, c->d_rot_y, amp, d_UB, d_EB));
    if (d_WB) PSE_TRY(pse_unpack(c, c->d_rot_y + half, amp, d_WB, nullptr));
    return st;
}

pse_status pse_step_full(pse_ctx *c, float *d_pos, double dt, const float *d_L, const float *d_noise_real, const float *d_noise_wave,
                         float *d_W, int *gmres_iters, int *lanczos_iters) {
    if (!c || !d_pos || !(dt > 0) || !d_noise_real || !d_noise_wave) return PSE_EINVAL;
    PSE_TRY(ensure_couplet(c));
    const int N = c->N, TB = 256, nb = (N + TB - 1) / TB;
    const float L = (float)c->L, invL = 1.0f / L;
    // [N][3] / [N][5] vectors in original numbering, carved out of the wide Lanczos vectors (idle outside pse_brownian_full)
    float *UB = c->d_rot_w, *EB = UB + (size_t)3 * N, *FP = UB + (size_t)8 * N, *U = UB + (size_t)11 * N;
    float *S = c->d_rot_u, *FB = S + (size_t)8 * N;
    float4 *xh = reinterpret_cast<float4 *>(c->d_rot_y);
    pse_status soft = PSE_OK;
    // (76) Brownian slip at x_k
    PSE_TRY(pse_neighbors(c, d_pos));
    pse_status st = pse_brownian(c, dt, d_noise_real, d_noise_wave, UB, EB, lanczos_iters);
    if (st == PSE_ENOCONV) soft = st; else if (st != PSE_OK) return st;
    // (77) mid-point
    k_advance_full<<<nb, TB, 0, c->stream>>>(reinterpret_cast<const float4 *>(d_pos), UB, (float)(0.5 * dt), L, invL, N, xh, c->deformed ? 0 : 1); KERNEL_CHECK(c);
    PSE_TRY(pse_neighbors(c, reinterpret_cast<const float *>(xh)));
    // (78) F^P (overlap + bond forces) and the torques at the mid-point; stresslet-constrained [U; Omega]
    PSE_TRY(pse_hard_sphere_forces(c, dt, FP));
    if (c->n_bonds) {
        PSE_TRY(pse_bond_forces(c, FB));
        PSE_TRY(pse_axpby(c, (size_t)3 * N, 1.f, FB, 1.f, FP));
    }
    st = pse_constrained_solve_full(c, FP, d_L, UB, EB, U, d_W, S, gmres_iters);
    if (st == PSE_ENOCONV) soft = st; else if (st != PSE_OK) return st;
    // (79) full step from x_k
    k_advance_full<<<nb, TB, 0, c->stream>>>(reinterpret_cast<const float4 *>(d_pos), U, (float)dt, L, invL, N, reinterpret_cast<float4 *>(d_pos),
                                             c->deformed ? 0 : 1); KERNEL_CHECK(c);
    return soft;
}

pse_status pse_mobility_apply_full(pse_ctx *c, const float *d_F, const float *d_L, const float *d_S, float *d_U, float *d_W, float *d_E, int which) {
    if (!c || !(which & PSE_BOTH) || (!d_F && !d_L && !d_S) || (!d_U && !d_W && !d_E)) return PSE_EINVAL;
    if (!c->have_nbrs) { c->err = "pse_mobility_apply_full before pse_neighbors"; return PSE_ENOTREADY; }
    if (!d_L && !d_W) return pse_mobility_apply(c, d_F, d_S, d_U, d_E, which);       // no torque in, no angular velocity out: the 8-component path
    PSE_TRY(ensure_couplet(c));
    PSE_TRY(pse_pack(c, d_F, d_S, c->d_in));
    PSE_TRY(pse_pack(c, d_L, nullptr, c->d_rot_in));
    PSE_TRY(apply_full_packed(c, c->d_in, c->d_rot_in, c->d_out, c->d_rot_out, which));
    if (d_U || d_E) PSE_TRY(pse_unpack(c, c->d_out, 1.f, d_U, d_E));
    if (d_W) PSE_TRY(pse_unpack(c, c->d_rot_out, 1.f, d_W, nullptr));
    return PSE_OK;
}

pse_status pse_constrained_solve_full(pse_ctx *c, const float *d_F, const float *d_L, const float *d_UB, const float *d_EB,
                                      float *d_U, float *d_W, float *d_S, int *gmres_iters) {
    if (!c || !d_U || !d_S) return PSE_EINVAL;
    if (!c->have_nbrs) { c->err = "pse_constrained_solve_full before pse_neighbors"; return PSE_ENOTREADY; }
    PSE_TRY(ensure_couplet(c));
    const size_t vec = (size_t)c->N * 8 * sizeof(float);
    PSE_TRY(pse_pack(c, d_UB, d_EB, c->d_vecB));
    PSE_TRY(pse_pack(c, d_L, nullptr, c->d_rot_in));
    if (d_L) {
        // what the torques alone do: (U_L, E_L) joins the Brownian slip on the right-hand side of Eq. (38)
        CUDA_TRY(c, cudaMemsetAsync(c->d_in, 0, vec, c->stream));
        PSE_TRY(apply_full_packed(c, c->d_in, c->d_rot_in, c->d_rot_tmp, c->d_rot_out, PSE_BOTH));
        PSE_TRY(pse_axpby(c, (size_t)c->N * 8, 1.f, c->d_rot_tmp, 1.f, c->d_vecB));
    }
    if (d_F) PSE_TRY(pse_pack(c, d_F, nullptr, c->d_vecA));
    pse_status st = pse_gmres_constraint(c, d_F ? c->d_vecA : nullptr, c->d_vecB, c->d_vecB, c->d_vecC, gmres_iters);
    if (st != PSE_OK && st != PSE_ENOCONV) return st;
    PSE_TRY(pse_unpack(c, c->d_vecC, 1.f, d_U, d_S));
    if (d_W) {                                                       // Omega = M_OF F + M_OL L + M_OS S: the Omega rows of one more full product
        k_merge_force_stresslet<<<(c->N + 255) / 256, 256, 0, c->stream>>>(d_F ? reinterpret_cast<const float4 *>(c->d_vecA) : nullptr,
                                                                           reinterpret_cast<const float4 *>(c->d_vecC), c->N, reinterpret_cast<float4 *>(c->d_in));
        KERNEL_CHECK(c);
        PSE_TRY(apply_full_packed(c, c->d_in, c->d_rot_in, c->d_out, c->d_rot_out, PSE_BOTH));
        PSE_TRY(pse_unpack(c, c->d_rot_out, 1.f, d_W, nullptr));
    }
    return st;
}

}  // extern "C"

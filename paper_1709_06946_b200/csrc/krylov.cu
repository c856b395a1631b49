// Device Krylov drivers (steps a8, a9): Lanczos for M_r^{1/2} w (Chow & Saad) and GMRES for the
// stresslet constraint M_ES S = -(E^B + M_EF F) (Eqs. 36-38, 78; 8-10 iterations,
// PAPER.md:561).  All vectors live on the device in the packed, cell-sorted layout [N][8] = (x,y,z,e1..e5); only
// the few scalars per iteration (dots, norms) cross to the host, where the tiny tridiagonal / Hessenberg work is
// done in fp64.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <cooperative_groups.h>
#include "pse_internal.h"

namespace cg = cooperative_groups;

namespace {

constexpr int VT = 256;
inline int vgrid(size_t n4) { size_t b = (n4 + VT - 1) / VT; return (int)(b < 1184 ? (b ? b : 1) : 1184); }   // 8 x 148

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[VT / 32];
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0;
    if (threadIdx.x < 32) {
        r = threadIdx.x < VT / 32 ? sh[threadIdx.x] : 0.0;
        for (int o = 16; o; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    __syncthreads();
    return r;
}

__global__ void k_pack(const float *F, const float *S, const int *order, int N, float4 *packed) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    int o = order[s];
    float f0 = 0, f1 = 0, f2 = 0, s0 = 0, s1 = 0, s2 = 0, s3 = 0, s4 = 0;
    if (F) { f0 = F[3 * o]; f1 = F[3 * o + 1]; f2 = F[3 * o + 2]; }
    if (S) { s0 = S[5 * o]; s1 = S[5 * o + 1]; s2 = S[5 * o + 2]; s3 = S[5 * o + 3]; s4 = S[5 * o + 4]; }
    packed[2 * s] = make_float4(f0, f1, f2, s0); packed[2 * s + 1] = make_float4(s1, s2, s3, s4);
}

__global__ void k_pack8(const float4 *v8, const int *order, int N, float4 *packed) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    int o = order[s];
    packed[2 * s] = v8[2 * o]; packed[2 * s + 1] = v8[2 * o + 1];
}

__global__ void k_unpack(const float4 *packed, const int *order, int N, float scale, float *U, float *E) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    int o = order[s];
    float4 a = packed[2 * s], b = packed[2 * s + 1];
    if (U) { U[3 * o] = scale * a.x; U[3 * o + 1] = scale * a.y; U[3 * o + 2] = scale * a.z; }
    if (E) { E[5 * o] = scale * a.w; E[5 * o + 1] = scale * b.x; E[5 * o + 2] = scale * b.y; E[5 * o + 3] = scale * b.z; E[5 * o + 4] = scale * b.w; }
}

// out[j] += <V_j, w>, j < nvec  (V_j = base + j*stride)
__global__ void __launch_bounds__(VT) k_multi_dot(const float4 *base, size_t stride4, int nvec, const float4 *w, size_t n4, double *out) {
    for (int j = 0; j < nvec; ++j) {
        const float4 *v = base + (size_t)j * stride4;
        double acc = 0;
        for (size_t i = (size_t)blockIdx.x * VT + threadIdx.x; i < n4; i += (size_t)gridDim.x * VT) {
            float4 a = v[i], b = w[i];
            acc += (double)(a.x * b.x + a.y * b.y) + (double)(a.z * b.z + a.w * b.w);
        }
        acc = block_sum(acc);
        if (threadIdx.x == 0) atomicAdd(out + j, acc);
    }
}


// out = beta * init + sum_j coef[j] V_j   (init may be null)
__global__ void __launch_bounds__(VT) k_lincomb(float4 *out, const float4 *init, float beta, const float4 *base, size_t stride4, int nvec,
                                                const float *coef, size_t n4) {
    for (size_t i = (size_t)blockIdx.x * VT + threadIdx.x; i < n4; i += (size_t)gridDim.x * VT) {
        float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
        if (init) { x = init[i]; x.x *= beta; x.y *= beta; x.z *= beta; x.w *= beta; }
        for (int j = 0; j < nvec; ++j) {
            float4 v = base[(size_t)j * stride4 + i]; float cj = coef[j];
            x.x += cj * v.x; x.y += cj * v.y; x.z += cj * v.z; x.w += cj * v.w;
        }
        out[i] = x;
    }
}

// y = alpha x + beta y
__global__ void __launch_bounds__(VT) k_axpby(size_t n, float alpha, const float *x, float beta, float *y) {
    for (size_t i = (size_t)blockIdx.x * VT + threadIdx.x; i < n; i += (size_t)gridDim.x * VT)
        y[i] = alpha * x[i] + (beta != 0.f ? beta * y[i] : 0.f);
}


// rhs = -(EB + E-part(z0)) embedded with zero velocity components (either input may be null)
__global__ void __launch_bounds__(VT) k_rhs(float4 *dst, const float4 *EBp, const float4 *z0, int N) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    float4 a = make_float4(0, 0, 0, 0), b = a;
    if (EBp) { a = EBp[2 * s]; b = EBp[2 * s + 1]; }
    if (z0) { float4 c = z0[2 * s], d = z0[2 * s + 1]; a.w += c.w; b.x += d.x; b.y += d.y; b.z += d.z; b.w += d.w; }
    dst[2 * s] = make_float4(0.f, 0.f, 0.f, -a.w);
    dst[2 * s + 1] = make_float4(-b.x, -b.y, -b.z, -b.w);
}

// out = ( U^B + U-rows of Zfin ; S-rows of fin )
__global__ void __launch_bounds__(VT) k_constraint_result(float4 *out, const float4 *UBp, const float4 *Zfin, const float4 *fin, int N) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    float ux = 0, uy = 0, uz = 0;
    if (UBp) { const float4 a = UBp[2 * s]; ux = a.x; uy = a.y; uz = a.z; }
    if (Zfin) { const float4 a = Zfin[2 * s]; ux += a.x; uy += a.y; uz += a.z; }
    const float4 fa = fin[2 * s], fb = fin[2 * s + 1];
    out[2 * s] = make_float4(ux, uy, uz, fa.w); out[2 * s + 1] = fb;
}

// ---- device-resident scalars: the update kernels read alpha / beta / h straight from the slots the dot kernels
// accumulated into, so an iteration needs one host read-back (for the tiny T / Hessenberg algebra and the stopping
// test) instead of a read-back plus a coefficient upload per reduction. ----

// dst = src / sqrt(*norm2)   (dst = 0 if the norm vanishes)
__global__ void __launch_bounds__(VT) k_scale_dev(float4 *dst, const float4 *src, const double *norm2, size_t n4) {
    const double n2 = *norm2;
    const float sc = n2 > 0 ? (float)(1.0 / sqrt(n2)) : 0.f;
    for (size_t i = (size_t)blockIdx.x * VT + threadIdx.x; i < n4; i += (size_t)gridDim.x * VT) {
        float4 x = src[i];
        x.x *= sc; x.y *= sc; x.z *= sc; x.w *= sc;
        dst[i] = x;
    }
}

// ---- one cooperative launch per Krylov iteration: the three dependent vector passes (dots, update + norm, scale)
// are separated by grid barriers instead of kernel boundaries; the vectors (2 MB at N = 65536) stay in L2 ----

// Lanczos:  alpha = <v_j, u>;  u -= alpha v_j + beta_{j-1} v_{j-1};  beta_j^2 = |u|^2;  v_{j+1} = u / beta_j
__global__ void __launch_bounds__(VT) k_lanczos_step(float4 *u, const float4 *vj, const float4 *vjm1, float4 *vnext, double *alpha,
                                                     const double *beta2_prev, double *beta2_out, size_t n4) {
    cg::grid_group grid = cg::this_grid();
    const size_t i0 = (size_t)blockIdx.x * VT + threadIdx.x, step = (size_t)gridDim.x * VT;
    double acc = 0;
    for (size_t i = i0; i < n4; i += step) {
        const float4 a = vj[i], b = u[i];
        acc += (double)(a.x * b.x + a.y * b.y) + (double)(a.z * b.z + a.w * b.w);
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) atomicAdd(alpha, acc);
    grid.sync();
    const float a = (float)*alpha, b = beta2_prev ? (float)sqrt(*beta2_prev) : 0.f;
    acc = 0;
    for (size_t i = i0; i < n4; i += step) {
        float4 x = u[i];
        const float4 v = vj[i];
        x.x -= a * v.x; x.y -= a * v.y; x.z -= a * v.z; x.w -= a * v.w;
        if (vjm1) { const float4 p = vjm1[i]; x.x -= b * p.x; x.y -= b * p.y; x.z -= b * p.z; x.w -= b * p.w; }
        u[i] = x;
        acc += (double)(x.x * x.x + x.y * x.y) + (double)(x.z * x.z + x.w * x.w);
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) atomicAdd(beta2_out, acc);
    if (!vnext) return;                                       // uniform over the grid
    grid.sync();
    const double n2 = *beta2_out;
    const float sc = n2 > 0 ? (float)(1.0 / sqrt(n2)) : 0.f;
    for (size_t i = i0; i < n4; i += step) {
        float4 x = u[i];                                      // this thread's own writes of the pass above
        x.x *= sc; x.y *= sc; x.z *= sc; x.w *= sc;
        vnext[i] = x;
    }
}

// Arnoldi:  h_j = <V_j, Z> (j < nvec);  w = Epart(Z) - sum_j h_j V_j;  h_{nvec} = |w|^2;  V_{nvec} = w / |w|
__global__ void __launch_bounds__(VT) k_arnoldi_step(float4 *w, const float4 *Z, const float4 *V, size_t stride4, int nvec, double *h,
                                                     float4 *vnext, int N) {
    cg::grid_group grid = cg::this_grid();
    const int s0 = blockIdx.x * VT + threadIdx.x, step = gridDim.x * VT;
    for (int j0 = 0; j0 < nvec; j0 += 4) {                   // four dots per pass over Z
        double acc[4] = {0, 0, 0, 0};
        for (int s = s0; s < N; s += step) {
            const float4 za = Z[2 * s], zb = Z[2 * s + 1];
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                if (j0 + jj < nvec) {
                    const float4 va = V[(size_t)(j0 + jj) * stride4 + 2 * s], vb = V[(size_t)(j0 + jj) * stride4 + 2 * s + 1];
                    acc[jj] += (double)(va.x * za.x + va.y * za.y) + (double)(va.z * za.z + va.w * za.w)
                             + (double)(vb.x * zb.x + vb.y * zb.y) + (double)(vb.z * zb.z + vb.w * zb.w);
                }
            }
        }
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            if (j0 + jj < nvec) { const double r = block_sum(acc[jj]); if (threadIdx.x == 0) atomicAdd(h + j0 + jj, r); }
        }
    }
    grid.sync();
    double acc = 0;
    for (int s = s0; s < N; s += step) {
        float4 a = Z[2 * s], b = Z[2 * s + 1];
        a.x = a.y = a.z = 0.f;
        for (int j = 0; j < nvec; ++j) {
            const float hj = (float)h[j];
            const float4 va = V[(size_t)j * stride4 + 2 * s], vb = V[(size_t)j * stride4 + 2 * s + 1];
            a.w -= hj * va.w; b.x -= hj * vb.x; b.y -= hj * vb.y; b.z -= hj * vb.z; b.w -= hj * vb.w;
        }
        w[2 * s] = a; w[2 * s + 1] = b;
        acc += (double)(a.w * a.w + b.x * b.x) + (double)(b.y * b.y + b.z * b.z) + (double)(b.w * b.w);
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) atomicAdd(h + nvec, acc);
    if (!vnext) return;
    grid.sync();
    const double n2 = h[nvec];
    const float sc = n2 > 0 ? (float)(1.0 / sqrt(n2)) : 0.f;
    for (int s = s0; s < N; s += step) {
        float4 a = w[2 * s], b = w[2 * s + 1];
        a.x *= sc; a.y *= sc; a.z *= sc; a.w *= sc; b.x *= sc; b.y *= sc; b.z *= sc; b.w *= sc;
        vnext[2 * s] = a; vnext[2 * s + 1] = b;
    }
}

// ---- the small algebra of a solve with a FIXED iteration count, on the device (one warp), so that the host need not be in
// the loop: pse_step enqueues both solves with the counts the previous step needed and looks at the scalars only afterwards ----

// coef[0..m) = |w| T_m^{1/2} e_1 for the Lanczos tridiagonal T_m (alpha_j on the diagonal, beta_j next to it), by the implicit
// QL iteration with Wilkinson shift (EISPACK imtql2).  Every lane carries its own copy of (d, e) and runs the scalar recurrence
// redundantly (identical values, no exchange, no barrier); lane k accumulates row k (and k + 32) of the eigenvector matrix.
// scal: [0] = |w|^2, [1 + 2j] = alpha_j, [2 + 2j] = beta_j^2.
__global__ void __launch_bounds__(32) k_lanczos_coef_dev(const double *__restrict__ scal, int m, float *__restrict__ coef) {
    __shared__ double z0[PSE_MAX_KRYLOV];                 // row 0 of the eigenvector matrix (first components), for the last step
    double d[PSE_MAX_KRYLOV], e[PSE_MAX_KRYLOV], za[PSE_MAX_KRYLOV], zb[PSE_MAX_KRYLOV];
    const int lane = threadIdx.x;
    for (int i = 0; i < m; ++i) {
        d[i] = scal[1 + 2 * i]; e[i] = i + 1 < m ? sqrt(fmax(scal[2 + 2 * i], 0.0)) : 0.0;
        za[i] = i == lane ? 1.0 : 0.0; zb[i] = i == lane + 32 ? 1.0 : 0.0;
    }
    for (int l = 0; l < m; ++l) {
        for (int iter = 0; iter < 60; ++iter) {
            int mm = l;
            for (; mm < m - 1; ++mm) { const double dd = fabs(d[mm]) + fabs(d[mm + 1]); if (fabs(e[mm]) <= 2e-16 * dd) break; }
            if (mm == l) break;
            double g = (d[l + 1] - d[l]) / (2.0 * e[l]), r = sqrt(g * g + 1.0);
            g = d[mm] - d[l] + e[l] / (g + (g >= 0 ? r : -r));
            double sn = 1.0, cs = 1.0, pp = 0.0;
            int i = mm - 1;
            bool under = false;
            for (; i >= l; --i) {
                double f = sn * e[i];
                const double b = cs * e[i];
                r = sqrt(f * f + g * g);
                e[i + 1] = r;
                if (r == 0.0) { d[i + 1] -= pp; e[mm] = 0.0; under = true; break; }
                const double ir = 1.0 / r;
                sn = f * ir; cs = g * ir;
                g = d[i + 1] - pp;
                r = (d[i] - g) * sn + 2.0 * cs * b;
                pp = sn * r;
                d[i + 1] = g + pp;
                g = cs * r - b;
                f = za[i + 1]; za[i + 1] = sn * za[i] + cs * f; za[i] = cs * za[i] - sn * f;        // my rows of the eigenvectors
                if (m > 32) { f = zb[i + 1]; zb[i + 1] = sn * zb[i] + cs * f; zb[i] = cs * zb[i] - sn * f; }
            }
            if (under) continue;
            d[l] -= pp; e[l] = g; e[mm] = 0.0;
        }
    }
    if (lane == 0) for (int k = 0; k < m; ++k) z0[k] = za[k];
    __syncwarp();
    const double wn = sqrt(fmax(scal[0], 0.0));
    for (int half = 0; half < 2; ++half) {
        const int i = lane + 32 * half;
        if (i >= m) break;
        double acc = 0.0;
        for (int k = 0; k < m; ++k) acc += (half ? zb[k] : za[k]) * sqrt(fmax(d[k], 0.0)) * z0[k];
        coef[i] = (float)(wn * acc);
    }
}

// y[0..m) of the GMRES least-squares problem after m Arnoldi iterations: Givens rotations column by column, back-substitution.
// scal: [0] = |b|^2; iteration k owns [base_k .. base_k + k + 1] = h_0..h_k, |w|^2 with base_k = 1 + k(k+3)/2.
__global__ void __launch_bounds__(32) k_gmres_coef_dev(const double *__restrict__ scal, int m, float *__restrict__ coef) {
    __shared__ double H[PSE_MAX_KRYLOV + 1][PSE_MAX_KRYLOV], cs[PSE_MAX_KRYLOV], sn[PSE_MAX_KRYLOV], g[PSE_MAX_KRYLOV + 1], y[PSE_MAX_KRYLOV];
    if (threadIdx.x != 0) return;
    g[0] = sqrt(fmax(scal[0], 0.0));
    for (int e = 0; e < m; ++e) {
        const int eb = 1 + e * (e + 3) / 2;
        for (int j = 0; j <= e; ++j) H[j][e] = scal[eb + j];
        H[e + 1][e] = sqrt(fmax(scal[eb + e + 1], 0.0));
        for (int j = 0; j < e; ++j) {
            const double a = H[j][e], b = H[j + 1][e];
            H[j][e] = cs[j] * a + sn[j] * b; H[j + 1][e] = -sn[j] * a + cs[j] * b;
        }
        const double a = H[e][e], b = H[e + 1][e], r = hypot(a, b);
        cs[e] = r > 0 ? a / r : 1.0; sn[e] = r > 0 ? b / r : 0.0;
        H[e][e] = r; H[e + 1][e] = 0.0;
        g[e + 1] = -sn[e] * g[e]; g[e] = cs[e] * g[e];
    }
    for (int i = m - 1; i >= 0; --i) {
        double s = g[i];
        for (int j = i + 1; j < m; ++j) s -= H[i][j] * y[j];
        y[i] = H[i][i] != 0.0 ? s / H[i][i] : 0.0;
    }
    for (int i = 0; i < m; ++i) coef[i] = (float)y[i];
}

// grid of a cooperative launch: every CTA must be resident (cap computed per device in pse_krylov_init)
int coop_grid(const pse_ctx *c, size_t work_items) {
    const size_t b = (work_items + 2 * VT - 1) / (2 * VT);          // at least two items per thread: fewer CTAs at the barriers
    return (int)std::max<size_t>(1, std::min<size_t>(b, (size_t)c->coop_cap));
}

// cyclic Jacobi eigen-decomposition of a small symmetric matrix (n <= 51), fp64, host
void jacobi_eigh(int n, std::vector<double> &A, std::vector<double> &Q) {
    Q.assign((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) Q[(size_t)i * n + i] = 1.0;
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0;
        for (int p = 0; p < n; ++p) for (int q = p + 1; q < n; ++q) off += A[(size_t)p * n + q] * A[(size_t)p * n + q];
        if (off < 1e-30) break;
        for (int p = 0; p < n; ++p) for (int q = p + 1; q < n; ++q) {
            double apq = A[(size_t)p * n + q];
            if (std::fabs(apq) < 1e-300) continue;
            double th = (A[(size_t)q * n + q] - A[(size_t)p * n + p]) / (2 * apq);
            double t = (th >= 0 ? 1.0 : -1.0) / (std::fabs(th) + std::sqrt(th * th + 1)), cs = 1 / std::sqrt(t * t + 1), sn = t * cs;
            for (int k = 0; k < n; ++k) {
                double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
                A[(size_t)k * n + p] = cs * akp - sn * akq; A[(size_t)k * n + q] = sn * akp + cs * akq;
            }
            for (int k = 0; k < n; ++k) {
                double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
                A[(size_t)p * n + k] = cs * apk - sn * aqk; A[(size_t)q * n + k] = sn * apk + cs * aqk;
            }
            for (int k = 0; k < n; ++k) {
                double qkp = Q[(size_t)k * n + p], qkq = Q[(size_t)k * n + q];
                Q[(size_t)k * n + p] = cs * qkp - sn * qkq; Q[(size_t)k * n + q] = sn * qkp + cs * qkq;
            }
        }
    }
}

pse_status read_scalars(pse_ctx *c, int n) {
    CUDA_TRY(c, cudaMemcpyAsync(c->h_scal, c->d_scal, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return PSE_OK;
}
pse_status zero_scalars(pse_ctx *c, int n) {
    CUDA_TRY(c, cudaMemsetAsync(c->d_scal, 0, (size_t)n * sizeof(double), c->stream));
    return PSE_OK;
}
pse_status upload_coefs(pse_ctx *c, const std::vector<float> &v) {
    float *hp = reinterpret_cast<float *>(c->h_scal + 2048);
    std::memcpy(hp, v.data(), v.size() * sizeof(float));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_coef, hp, v.size() * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    return PSE_OK;
}

}  // namespace

pse_status pse_krylov_init(pse_ctx *c) {
    int a = 0, b = 0, coop = 0;
    CUDA_TRY(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device));
    if (!coop) { c->err = "device does not support cooperative launches (Krylov step kernels)"; return PSE_ECUDA; }
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, k_lanczos_step, VT, 0));
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_arnoldi_step, VT, 0));
    c->coop_cap = c->nsm * std::max(1, std::min(a, b));
    return PSE_OK;
}

pse_status pse_pack(pse_ctx *c, const float *d_F, const float *d_S, float *d_packed) {
    ScopedPhase ph(c, PSE_T_PACK);
    k_pack<<<(c->N + VT - 1) / VT, VT, 0, c->stream>>>(d_F, d_S, c->d_order, c->N, reinterpret_cast<float4 *>(d_packed)); KERNEL_CHECK(c);
    return PSE_OK;
}
pse_status pse_pack8(pse_ctx *c, const float *d_v8, float *d_packed) {
    ScopedPhase ph(c, PSE_T_PACK);
    k_pack8<<<(c->N + VT - 1) / VT, VT, 0, c->stream>>>(reinterpret_cast<const float4 *>(d_v8), c->d_order, c->N, reinterpret_cast<float4 *>(d_packed)); KERNEL_CHECK(c);
    return PSE_OK;
}
pse_status pse_unpack(pse_ctx *c, const float *d_packed, float scale, float *d_U, float *d_E) {
    ScopedPhase ph(c, PSE_T_PACK);
    k_unpack<<<(c->N + VT - 1) / VT, VT, 0, c->stream>>>(reinterpret_cast<const float4 *>(d_packed), c->d_order, c->N, scale, d_U, d_E); KERNEL_CHECK(c);
    return PSE_OK;
}
pse_status pse_axpby(pse_ctx *c, size_t n, float alpha, const float *x, float beta, float *y) {
    ScopedPhase ph(c, PSE_T_VECTOR);
    k_axpby<<<vgrid(n), VT, 0, c->stream>>>(n, alpha, x, beta, y); KERNEL_CHECK(c);
    return PSE_OK;
}

// y = M_r^{1/2} w  by Lanczos:  v_1 = w/|w|,  T_m = V_m^T M_r V_m,  y_m = |w| V_m T_m^{1/2} e_1.
// Stop when |y_m - y_{m-1}| <= tol |y_m|; with V orthonormal this is the change of the coefficient vector.
// fixed_m > 0: exactly fixed_m iterations, coefficients by k_lanczos_coef_dev, no host read-back: the scalars are copied to
// h_scal_l behind the solve and examined by pse_lanczos_validate once the stream has been synchronised.
static pse_status real_apply_all(pse_ctx *c, const float *d_in, float *d_out) { return pse_real_apply(c, d_in, d_out); }
static pse_status lanczos_impl(pse_ctx *c, const float *d_w, float *d_y, int *iters, int fixed_m, int width, pse_matvec_fn op, float *d_u);

pse_status pse_lanczos_sqrt(pse_ctx *c, const float *d_w, float *d_y, int *iters, int fixed_m) {
    return lanczos_impl(c, d_w, d_y, iters, fixed_m, 1, real_apply_all, c->d_tmp);
}
pse_status pse_lanczos_sqrt_wide(pse_ctx *c, const float *d_w, float *d_y, int *iters, int width, pse_matvec_fn op, float *d_u) {
    return lanczos_impl(c, d_w, d_y, iters, 0, width, op, d_u);
}

static pse_status lanczos_impl(pse_ctx *c, const float *d_w, float *d_y, int *iters, int fixed_m, int width, pse_matvec_fn op, float *d_u) {
    const size_t n = (size_t)c->N * 8 * width, n4 = n / 4;
    float4 *V = reinterpret_cast<float4 *>(c->d_krylov);
    float4 *u = reinterpret_cast<float4 *>(d_u);
    const int maxit = std::min(PSE_MAX_KRYLOV, c->krylov_cap / width - 1);
    // slots: [0] = |w|^2, [1+2j] = alpha_j, [2+2j] = beta_j^2
    const int nslots = 1 + 2 * maxit;
    PSE_TRY(zero_scalars(c, nslots));
    { ScopedPhase ph(c, PSE_T_VECTOR);
      k_multi_dot<<<vgrid(n4), VT, 0, c->stream>>>(reinterpret_cast<const float4 *>(d_w), 0, 1, reinterpret_cast<const float4 *>(d_w), n4, c->d_scal); KERNEL_CHECK(c);
      k_scale_dev<<<vgrid(n4), VT, 0, c->stream>>>(V, reinterpret_cast<const float4 *>(d_w), c->d_scal, n4); KERNEL_CHECK(c); }
    if (iters) *iters = 0;
    std::vector<double> alpha, beta, cprev, ccur;
    double wn = 0;
    int m = 0;
    bool converged = false;
    // The host only decides when to stop, so it need not look at every iteration: the read-back (a stream
    // synchronisation that idles the GPU) is skipped until one iteration before the count the previous call needed;
    // the skipped iterations are then examined in order and the first converged one is taken — same result as
    // checking every time.
    // (once the count has repeated, only the iteration it is expected to end in is read back: one synchronisation per solve)
    const int first_check = width > 1 ? 0 : std::max(0, c->last_lanczos_iters - (c->lanczos_repeats >= 2 ? 1 : 2));
    int examined = 0;
    const int niter = fixed_m > 0 ? std::min(fixed_m, maxit) : maxit;
    for (int j = 0; j < niter && !converged; ++j) {
        float4 *vj = V + (size_t)j * n4;
        PSE_TRY(op(c, reinterpret_cast<const float *>(vj), reinterpret_cast<float *>(u)));
        { ScopedPhase ph(c, PSE_T_VECTOR);
          const float4 *a_vj = vj, *a_vjm1 = j ? vj - n4 : nullptr;
          float4 *a_u = u, *a_next = j + 1 < niter ? vj + n4 : nullptr;
          double *a_alpha = c->d_scal + 1 + 2 * j, *a_b2 = c->d_scal + 2 + 2 * j;
          const double *a_b2prev = j ? c->d_scal + 2 * j : nullptr;
          size_t a_n4 = n4;
          void *args[] = {&a_u, &a_vj, &a_vjm1, &a_next, &a_alpha, &a_b2prev, &a_b2, &a_n4};
          CUDA_TRY(c, cudaLaunchCooperativeKernel((const void *)k_lanczos_step, dim3(coop_grid(c, n4)), dim3(VT), args, 0, c->stream));
          KERNEL_CHECK(c); }
        if (fixed_m > 0) continue;
        if (j < first_check && j + 1 < maxit) continue;
        PSE_TRY(read_scalars(c, 3 + 2 * j));
        for (; examined <= j && !converged; ++examined) {
            const int e_j = examined;
            if (e_j == 0) {
                wn = std::sqrt(c->h_scal[0]);
                if (!(wn > 0)) { CUDA_TRY(c, cudaMemsetAsync(d_y, 0, n * sizeof(float), c->stream)); return PSE_OK; }
            }
            alpha.push_back(c->h_scal[1 + 2 * e_j]);
            beta.push_back(std::sqrt(c->h_scal[2 + 2 * e_j]));
            m = e_j + 1;
            // coefficient vector  c = |w| T^{1/2} e_1  of the m x m tridiagonal
            std::vector<double> Tm((size_t)m * m, 0.0), Q;
            for (int i = 0; i < m; ++i) { Tm[(size_t)i * m + i] = alpha[i]; if (i + 1 < m) Tm[(size_t)i * m + i + 1] = Tm[(size_t)(i + 1) * m + i] = beta[i]; }
            jacobi_eigh(m, Tm, Q);
            ccur.assign(m, 0.0);
            for (int e = 0; e < m; ++e) {
                double lam = Tm[(size_t)e * m + e], sq = lam > 0 ? std::sqrt(lam) : 0.0, q0 = Q[e];       // Q[0][e]
                for (int i = 0; i < m; ++i) ccur[i] += wn * Q[(size_t)i * m + e] * sq * q0;
            }
            double diff = 0, nrm = 0;
            for (int i = 0; i < m; ++i) { double d = ccur[i] - (i < (int)cprev.size() ? cprev[i] : 0.0); diff += d * d; nrm += ccur[i] * ccur[i]; }
            cprev = ccur;
            if (e_j > 0 && std::sqrt(diff) <= c->tol * std::sqrt(nrm)) converged = true;
            else if (beta[e_j] <= 1e-7 * std::fabs(alpha[0])) converged = true;                          // invariant subspace
        }
    }
    if (fixed_m > 0) {
        k_lanczos_coef_dev<<<1, 32, 0, c->stream>>>(c->d_scal, niter, c->d_coef); KERNEL_CHECK(c);
        { ScopedPhase ph(c, PSE_T_VECTOR);
          k_lincomb<<<vgrid(n4), VT, 0, c->stream>>>(reinterpret_cast<float4 *>(d_y), nullptr, 0.f, V, n4, niter, c->d_coef, n4); KERNEL_CHECK(c); }
        CUDA_TRY(c, cudaMemcpyAsync(c->h_scal_l, c->d_scal, (size_t)(1 + 2 * niter) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        if (iters) *iters = niter;
        return PSE_OK;
    }
    if (width == 1) {
        c->lanczos_repeats = (m == c->last_lanczos_iters) ? c->lanczos_repeats + 1 : 0;
        c->last_lanczos_iters = m;
    }
    std::vector<float> cf(ccur.begin(), ccur.end());
    PSE_TRY(upload_coefs(c, cf));
    { ScopedPhase ph(c, PSE_T_VECTOR);
      k_lincomb<<<vgrid(n4), VT, 0, c->stream>>>(reinterpret_cast<float4 *>(d_y), nullptr, 0.f, V, n4, m, c->d_coef, n4); KERNEL_CHECK(c); }
    if (iters) *iters = m;
    if (!converged) { c->err = "Lanczos did not converge"; return PSE_ENOCONV; }
    return PSE_OK;
}

// coefficient vector |w| T_m^{1/2} e_1 of the leading m x m block, host fp64 (Jacobi)
static std::vector<double> lanczos_coefs_host(const double *hs, int m) {
    std::vector<double> Tm((size_t)m * m, 0.0), Q, out(m, 0.0);
    for (int i = 0; i < m; ++i) {
        Tm[(size_t)i * m + i] = hs[1 + 2 * i];
        if (i + 1 < m) Tm[(size_t)i * m + i + 1] = Tm[(size_t)(i + 1) * m + i] = std::sqrt(std::max(hs[2 + 2 * i], 0.0));
    }
    jacobi_eigh(m, Tm, Q);
    const double wn = std::sqrt(std::max(hs[0], 0.0));
    for (int e = 0; e < m; ++e) {
        const double lam = Tm[(size_t)e * m + e], sq = lam > 0 ? std::sqrt(lam) : 0.0, q0 = Q[e];
        for (int i = 0; i < m; ++i) out[i] += wn * Q[(size_t)i * m + e] * sq * q0;
    }
    return out;
}

// After a fixed-count solve and a stream synchronisation: did the sample converge within m iterations (same criterion as the
// adaptive driver, |c_m - c_{m-1}| <= tol |c_m|), and would one iteration fewer have done (*shrink)?
bool pse_lanczos_validate(pse_ctx *c, int m, bool *shrink) {
    const double *hs = c->h_scal_l;
    *shrink = false;
    if (!(hs[0] > 0)) return true;                                   // zero noise: zero sample
    if (m < 2) return false;
    auto change = [&](int mm) {
        const std::vector<double> a = lanczos_coefs_host(hs, mm), b = lanczos_coefs_host(hs, mm - 1);
        double diff = 0, nrm = 0;
        for (int i = 0; i < mm; ++i) { const double d = a[i] - (i < mm - 1 ? b[i] : 0.0); diff += d * d; nrm += a[i] * a[i]; }
        return std::sqrt(diff) <= c->tol * std::sqrt(nrm);
    };
    const bool ok = change(m) || std::sqrt(std::max(hs[2 + 2 * (m - 1)], 0.0)) <= 1e-7 * std::fabs(hs[1]);
    if (ok && m >= 3) *shrink = change(m - 1);
    return ok;
}

// Same for GMRES: relative residual of the Givens recurrence after m iterations <= tol, and after m - 1 (*shrink).
bool pse_gmres_validate(pse_ctx *c, int m, bool *shrink) {
    const double *hs = c->h_scal;
    *shrink = false;
    const double bnorm = std::sqrt(std::max(hs[0], 0.0));
    if (!(bnorm > 0)) return true;
    std::vector<double> H((size_t)(m + 1) * m, 0.0), cs(m, 0.0), sn(m, 0.0), g(m + 1, 0.0);
    g[0] = bnorm;
    for (int e = 0; e < m; ++e) {
        const int eb = 1 + e * (e + 3) / 2;
        for (int j = 0; j <= e; ++j) H[(size_t)j * m + e] = hs[eb + j];
        H[(size_t)(e + 1) * m + e] = std::sqrt(std::max(hs[eb + e + 1], 0.0));
        for (int j = 0; j < e; ++j) {
            const double a = H[(size_t)j * m + e], b = H[(size_t)(j + 1) * m + e];
            H[(size_t)j * m + e] = cs[j] * a + sn[j] * b; H[(size_t)(j + 1) * m + e] = -sn[j] * a + cs[j] * b;
        }
        const double a = H[(size_t)e * m + e], b = H[(size_t)(e + 1) * m + e], r = std::hypot(a, b);
        cs[e] = r > 0 ? a / r : 1.0; sn[e] = r > 0 ? b / r : 0.0;
        g[e + 1] = -sn[e] * g[e]; g[e] = cs[e] * g[e];
        if (e + 1 == m - 1 && std::fabs(g[e + 1]) <= c->tol * bnorm) *shrink = true;
    }
    return std::fabs(g[m]) <= c->tol * bnorm;
}

// Forward declaration of the full product on packed vectors (api.cu)
pse_status pse_apply_packed(pse_ctx *c, const float *d_in, float *d_out, int which, int mode = PSE_MODE_ALL);

// GMRES on  M_ES S = -(E^B + M_EF F)  with S and E embedded in packed vectors whose velocity slots are zero.
// Z_j = M [0; v_j] is kept whole: its E-part feeds Arnoldi, its U-part gives M_US S at the end without another
// product.  out (packed) = (U, S) with U = U^B + M_UF F + M_US S.
pse_status pse_gmres_constraint(pse_ctx *c, const float *d_Fp, const float *d_UBp, const float *d_EBp, float *d_outp, int *iters, int fixed_m) {
    const int N = c->N;
    const size_t n = (size_t)N * 8, n4 = n / 4;
    float4 *V = reinterpret_cast<float4 *>(c->d_krylov), *Z = reinterpret_cast<float4 *>(c->d_zu);
    float4 *w = reinterpret_cast<float4 *>(c->d_tmp), *z0 = reinterpret_cast<float4 *>(c->d_tmp2);
    const int maxit = std::min(PSE_MAX_KRYLOV, c->krylov_cap - 1), nbN = (N + VT - 1) / VT;
    if (iters) *iters = 0;
    if (d_Fp) PSE_TRY(pse_apply_packed(c, d_Fp, reinterpret_cast<float *>(z0), PSE_BOTH, PSE_IN_F | PSE_OUT_E));     // M_EF F
    { ScopedPhase ph(c, PSE_T_VECTOR);
      k_rhs<<<nbN, VT, 0, c->stream>>>(w, reinterpret_cast<const float4 *>(d_EBp), d_Fp ? z0 : nullptr, N); KERNEL_CHECK(c); }
    // slots: [0] = |b|^2; iteration k owns [base_k .. base_k + k + 1] = h_0..h_k, |w|^2 with base_k = 1 + k(k+3)/2
    const int nslots = 1 + maxit * (maxit + 3) / 2;
    PSE_TRY(zero_scalars(c, nslots));
    { ScopedPhase ph(c, PSE_T_VECTOR);
      k_multi_dot<<<vgrid(n4), VT, 0, c->stream>>>(w, 0, 1, w, n4, c->d_scal); KERNEL_CHECK(c);
      k_scale_dev<<<vgrid(n4), VT, 0, c->stream>>>(V, w, c->d_scal, n4); KERNEL_CHECK(c); }
    double bnorm = 0;                                               // |b| arrives with the first read-back
    int m = 0;
    std::vector<double> H((size_t)(maxit + 1) * maxit, 0.0), cs(maxit, 0.0), sn(maxit, 0.0), g(maxit + 1, 0.0), y;
    bool converged = false;
    {
        const int first_check = std::max(0, c->last_gmres_iters - (c->gmres_repeats >= 2 ? 1 : 2));     // see pse_lanczos_sqrt
        int examined = 0;
        const int niter = fixed_m > 0 ? std::min(fixed_m, maxit) : maxit;
        for (int k = 0; k < niter && !converged; ++k) {
            const int base = 1 + k * (k + 3) / 2;
            float4 *Zk = Z + (size_t)k * n4;
            PSE_TRY(pse_apply_packed(c, reinterpret_cast<const float *>(V + (size_t)k * n4), reinterpret_cast<float *>(Zk), PSE_BOTH, PSE_IN_S | PSE_OUT_E));   // M_ES v_k: 5 grids in, 5 out
            { ScopedPhase ph(c, PSE_T_VECTOR);
              // the velocity slots of every V_j are zero, so <V_j, Z_k> over all 8 components is the E-part product
              float4 *a_w = w, *a_next = k + 1 < niter ? V + (size_t)(k + 1) * n4 : nullptr;
              const float4 *a_Z = Zk, *a_V = V;
              size_t a_stride = n4; int a_nvec = k + 1, a_N = N;
              double *a_h = c->d_scal + base;
              void *args[] = {&a_w, &a_Z, &a_V, &a_stride, &a_nvec, &a_h, &a_next, &a_N};
              CUDA_TRY(c, cudaLaunchCooperativeKernel((const void *)k_arnoldi_step, dim3(coop_grid(c, (size_t)N)), dim3(VT), args, 0, c->stream));
              KERNEL_CHECK(c); }
            if (fixed_m > 0) { m = k + 1; continue; }
            if (k < first_check && k + 1 < maxit) continue;
            PSE_TRY(read_scalars(c, base + k + 2));
            if (examined == 0) {
                bnorm = std::sqrt(c->h_scal[0]);
                if (!(bnorm > 0)) { converged = true; break; }          // zero right-hand side: S = 0
                g[0] = bnorm;
            }
            for (; examined <= k && !converged; ++examined) {
                const int e = examined, eb = 1 + e * (e + 3) / 2;
                for (int j = 0; j <= e; ++j) H[(size_t)j * maxit + e] = c->h_scal[eb + j];
                const double hk1 = std::sqrt(c->h_scal[eb + e + 1]);
                H[(size_t)(e + 1) * maxit + e] = hk1;
                for (int j = 0; j < e; ++j) {                        // apply previous Givens rotations to column e
                    double a = H[(size_t)j * maxit + e], b = H[(size_t)(j + 1) * maxit + e];
                    H[(size_t)j * maxit + e] = cs[j] * a + sn[j] * b; H[(size_t)(j + 1) * maxit + e] = -sn[j] * a + cs[j] * b;
                }
                double a = H[(size_t)e * maxit + e], b = H[(size_t)(e + 1) * maxit + e], r = std::hypot(a, b);
                cs[e] = r > 0 ? a / r : 1.0; sn[e] = r > 0 ? b / r : 0.0;
                H[(size_t)e * maxit + e] = r; H[(size_t)(e + 1) * maxit + e] = 0.0;
                g[e + 1] = -sn[e] * g[e]; g[e] = cs[e] * g[e];
                m = e + 1;
                if (std::fabs(g[e + 1]) <= c->tol * bnorm) converged = true;
                else if (hk1 <= 1e-12 * bnorm) converged = true;
            }
        }
        if (fixed_m > 0) {
            k_gmres_coef_dev<<<1, 32, 0, c->stream>>>(c->d_scal, m, c->d_coef); KERNEL_CHECK(c);
            CUDA_TRY(c, cudaMemcpyAsync(c->h_scal, c->d_scal, (size_t)(1 + m * (m + 3) / 2) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            converged = true;                                        // decided later by pse_gmres_validate
        } else {
            c->gmres_repeats = (m == c->last_gmres_iters) ? c->gmres_repeats + 1 : 0;
            c->last_gmres_iters = m;
        }
        y.assign(m, 0.0);
        for (int i = m - 1; i >= 0; --i) {
            double s = g[i];
            for (int j = i + 1; j < m; ++j) s -= H[(size_t)i * maxit + j] * y[j];
            y[i] = s / H[(size_t)i * maxit + i];
        }
    }
    // S = sum_j y_j v_j;  U = U^B + U-rows of M [F; S]: one last product with 3 output grids (the Arnoldi products
    // carried only the E rows)
    std::vector<float> yf(y.begin(), y.end());
    if (m && fixed_m <= 0) PSE_TRY(upload_coefs(c, yf));
    float4 *fin = w;                                               // [F; S] packed, reuses the Arnoldi work vector
    { ScopedPhase ph(c, PSE_T_VECTOR);
      k_lincomb<<<vgrid(n4), VT, 0, c->stream>>>(fin, reinterpret_cast<const float4 *>(d_Fp), 1.f, V, n4, m, c->d_coef, n4); KERNEL_CHECK(c); }
    const int fmode = (d_Fp ? PSE_IN_F : 0) | (m ? PSE_IN_S : 0) | PSE_OUT_U;
    if (fmode & (PSE_IN_F | PSE_IN_S)) PSE_TRY(pse_apply_packed(c, reinterpret_cast<const float *>(fin), reinterpret_cast<float *>(Z), PSE_BOTH, fmode));
    { ScopedPhase ph(c, PSE_T_VECTOR);
      k_constraint_result<<<nbN, VT, 0, c->stream>>>(reinterpret_cast<float4 *>(d_outp), reinterpret_cast<const float4 *>(d_UBp),
                                                     (fmode & (PSE_IN_F | PSE_IN_S)) ? Z : nullptr, fin, N); KERNEL_CHECK(c); }
    if (iters) *iters = m;
    if (!converged) { c->err = "GMRES did not converge"; return PSE_ENOCONV; }
    return PSE_OK;
}

// Own 3-D FFT for the wave-space sum, fused with the k-space scaling (steps a4-a6 of the path).
//
// cuFFT runs a 3-D R2C / C2R as three passes over the data each, and the scaling is a fourth and the middle of
// seven passes over the spectrum.  Here the transform is cut where the data is contiguous instead:
//
//   fft_fwd_plane_kernel   one CTA per (component, x-plane): the M x M real plane is loaded once, transformed along z
//                          (two real lines per complex FFT) and along y in shared memory, stored as M x Mhp complex.
//   fft_x_scale_kernel     one CTA per (ky, chunk of kz): all components' x-lines are loaded, transformed along x,
//                          multiplied by the k-space operator (the same code as scale_kernel: P^H B P), transformed
//                          back along x and stored.  The full spectrum never exists in memory.
//   fft_inv_plane_kernel   mirror image of the first.
//
// Three passes over the spectrum instead of seven.  Transforms are Stockham autosort stages between two shared-memory
// buffers; a stage's radix (2..5, or 6, 8, 9, 10, 12, 16 as two nested small transforms) is done in registers, so
// M = 100 takes two stages.  Lanes run over lines, so the twiddle of a butterfly is a broadcast and shared accesses
// are conflict-free (line index fastest-varying, or odd pitch).  Unnormalised like cuFFT.  The half-spectrum rows
// are padded to Mhp = 4*ceil(Mh/4) entries so that every row and every 8-entry chunk starts on a 32-byte sector.
// Sizes with other prime factors, or whose plane does not fit in shared memory, take the cuFFT path (wavespace.cu),
// which is also the default: see pse_fft_init for the measurements.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <string>
#include <vector>
#include "pse_internal.h"
#include "wave_scale.cuh"

namespace {

constexpr int FFT_THREADS = 512;
constexpr int XCH = 4;                           // kz entries per CTA of the x pass (one 32-byte sector per row)
constexpr int XT = 256;                          // threads of an x-pass CTA (four CTAs per SM)
constexpr int FFT_MAXSTAGE = 6;

// division by a run-time constant: q = floor(x / d) as one IMAD.HI; exact for x < 2^20, d <= 4096 (m = ceil(2^32 / d))
struct FastDiv {
    unsigned d, m;
    __device__ __forceinline__ int div(int x) const { return d == 1 ? x : (int)__umulhi((unsigned)x, m); }
};
inline FastDiv make_div(int d) { FastDiv f; f.d = (unsigned)d; f.m = d <= 1 ? 0u : (unsigned)((0x100000000ull + d - 1) / d); return f; }

struct FftStage { int R, Ns, nb, tstep; FastDiv ns_div; int pad[2]; };     // nb = M/R, tstep = M/(Ns R)

struct FftDev {                                  // lives in device memory (pse_ctx::d_fft_dev); kernels copy it to shared
    int M, Mh, Mhp, nstage;
    int Pz, PK, NP, bufsz;                       // odd pitch of the z-line buffer, pitch of the [y][kz] buffer (= Mhp), line pairs
    FastDiv divM, divMh, divNP, divMq;           // Mq = M/4 (float4 columns of a real row)
    FftStage st[FFT_MAXSTAGE];
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// multiplication by -i (forward) or +i (inverse)
template <bool INV> __device__ __forceinline__ float2 mul_mi(float2 a) { return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x); }
template <bool INV> __device__ __forceinline__ float2 twiddle(const float2 *tw, int idx) { float2 w = tw[idx]; if (INV) w.y = -w.y; return w; }

template <int R, bool INV> struct Bfly;
template <bool INV> struct Bfly<2, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[2]) { const float2 a = v[0], b = v[1]; v[0] = cadd(a, b); v[1] = csub(a, b); }
};
template <bool INV> struct Bfly<3, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[3]) {
        const float s = 0.86602540378443865f;
        const float2 t1 = cadd(v[1], v[2]), t2 = make_float2(v[0].x - 0.5f * t1.x, v[0].y - 0.5f * t1.y);
        const float2 d = csub(v[1], v[2]), t3 = mul_mi<INV>(make_float2(s * d.x, s * d.y));
        v[0] = cadd(v[0], t1); v[1] = cadd(t2, t3); v[2] = csub(t2, t3);
    }
};
template <bool INV> struct Bfly<4, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[4]) {
        const float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]), t2 = cadd(v[1], v[3]), t3 = mul_mi<INV>(csub(v[1], v[3]));
        v[0] = cadd(t0, t2); v[2] = csub(t0, t2); v[1] = cadd(t1, t3); v[3] = csub(t1, t3);
    }
};
template <bool INV> struct Bfly<5, INV> {
    static __device__ __forceinline__ void run(float2 (&v)[5]) {
        const float c1 = 0.30901699437494742f, s1 = 0.95105651629515357f, c2 = -0.80901699437494742f, s2 = 0.58778525229247313f;
        const float2 p1 = cadd(v[1], v[4]), m1 = csub(v[1], v[4]), p2 = cadd(v[2], v[3]), m2 = csub(v[2], v[3]);
        const float2 a = v[0];
        const float2 r1 = make_float2(a.x + c1 * p1.x + c2 * p2.x, a.y + c1 * p1.y + c2 * p2.y);
        const float2 r2 = make_float2(a.x + c2 * p1.x + c1 * p2.x, a.y + c2 * p1.y + c1 * p2.y);
        const float2 q1 = mul_mi<INV>(make_float2(s1 * m1.x + s2 * m2.x, s1 * m1.y + s2 * m2.y));
        const float2 q2 = mul_mi<INV>(make_float2(s2 * m1.x - s1 * m2.x, s2 * m1.y - s1 * m2.y));
        v[0] = make_float2(a.x + p1.x + p2.x, a.y + p1.y + p2.y);
        v[1] = cadd(r1, q1); v[4] = csub(r1, q1); v[2] = cadd(r2, q2); v[3] = csub(r2, q2);
    }
};

// DFT of size R1*R2 in registers, natural order in and out (Cooley-Tukey: R2 transforms of size R1 over stride R2,
// twiddles W_R^{n2 k1} = tw[n2 k1 M/R], R1 transforms of size R2).  wstep = M / R.
template <int R1, int R2, bool INV>
__device__ __forceinline__ void dft(float2 (&v)[R1 * R2], const float2 *tw, int wstep) {
    if constexpr (R2 == 1) {
        Bfly<R1, INV>::run(v);
    } else {
        float2 y[R1 * R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) {
            float2 t[R1];
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) t[n1] = v[R2 * n1 + n2];
            Bfly<R1, INV>::run(t);
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) y[n2 * R1 + k1] = (n2 && k1) ? cmul(t[k1], twiddle<INV>(tw, n2 * k1 * wstep)) : t[k1];
        }
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            float2 t[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) t[n2] = y[n2 * R1 + k1];
            Bfly<R2, INV>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) v[k1 + R1 * k2] = t[k2];
        }
    }
}

// One Stockham stage of radix R = R1*R2 over the lines l0 .. l0+nl-1; element i of line l sits at l*ls + i*es in src
// and dst.
template <int R1, int R2, bool INV, int NT>
__device__ __forceinline__ void stage(const float2 *__restrict__ src, float2 *__restrict__ dst, int l0, int nl, FastDiv nl_div, int ls, int es,
                                      const FftStage &S, const float2 *__restrict__ tw, int tid) {
    constexpr int R = R1 * R2;
    const int nb = S.nb, Ns = S.Ns, total = nl * nb, tstep = S.tstep, rs = nb * es, ws = Ns * es;
    const FastDiv ns_div = S.ns_div;
    for (int it = tid; it < total; it += NT) {
        const int j = nl_div.div(it), l = l0 + it - j * nl;         // lanes over lines
        const int q = ns_div.div(j), k = j - q * Ns;
        const float2 *s = src + l * ls + j * es;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = s[r * rs];
        if (k) {
            const int t1 = k * tstep;
#pragma unroll
            for (int r = 1; r < R; ++r) v[r] = cmul(v[r], twiddle<INV>(tw, r * t1));
        }
        dft<R1, R2, INV>(v, tw, nb);                                // M / R = nb
        float2 *d = dst + l * ls + (q * Ns * R + k) * es;
#pragma unroll
        for (int r = 0; r < R; ++r) d[r * ws] = v[r];
    }
}

// all stages; returns with the result in `a` (pointers are swapped as needed); ends with a barrier
template <bool INV, int NT>
__device__ __forceinline__ void fft_lines(float2 *&a, float2 *&b, const FftDev &f, int l0, int nl, FastDiv nl_div, int ls, int es,
                                          const float2 *tw, int tid) {
#pragma unroll 1
    for (int s = 0; s < f.nstage; ++s) {
        const FftStage &S = f.st[s];
#define PSE_STAGE(A, B) stage<A, B, INV, NT>(a, b, l0, nl, nl_div, ls, es, S, tw, tid)
        switch (S.R) {
            case 2: PSE_STAGE(2, 1); break;
            case 3: PSE_STAGE(3, 1); break;
            case 4: PSE_STAGE(4, 1); break;
            case 5: PSE_STAGE(5, 1); break;
            case 6: PSE_STAGE(3, 2); break;
            case 8: PSE_STAGE(4, 2); break;
            case 9: PSE_STAGE(3, 3); break;
            case 10: PSE_STAGE(5, 2); break;
            case 12: PSE_STAGE(4, 3); break;
            default: PSE_STAGE(4, 4); break;
        }
#undef PSE_STAGE
        __syncthreads();
        float2 *t = a; a = b; b = t;
    }
}

// shared-memory prologue common to the kernels: plan record, then twiddles (16-byte aligned), then the buffers
struct FftSmem { FftDev *f; float2 *tw, *A; };
template <int NT>
__device__ __forceinline__ FftSmem fft_prologue(unsigned char *raw, const FftDev *gf, const float2 *gtw, int tid) {
    FftSmem s;
    s.f = reinterpret_cast<FftDev *>(raw);
    constexpr int NW = (sizeof(FftDev) + 3) / 4, OFF = (sizeof(FftDev) + 15) / 16 * 16;
    for (int i = tid; i < NW; i += NT) reinterpret_cast<int *>(raw)[i] = reinterpret_cast<const int *>(gf)[i];
    s.tw = reinterpret_cast<float2 *>(raw + OFF);
    const int M = gf->M;
    for (int i = tid; i < M; i += NT) s.tw[i] = gtw[i];
    s.A = s.tw + ((M + 1) & ~1);
    return s;
}
inline size_t fft_prologue_bytes(int M) { return (sizeof(FftDev) + 15) / 16 * 16 + (size_t)((M + 1) & ~1) * sizeof(float2); }

// ---- forward: real [M][M] plane (y, z) -> complex [M][Mhp] (ky, kz) ----
__global__ void __launch_bounds__(FFT_THREADS, 2) fft_fwd_plane_kernel(const float *__restrict__ grid, float2 *__restrict__ spec,
                                                                       const FftDev *__restrict__ gf, const float2 *__restrict__ gtw, int first) {
    extern __shared__ __align__(16) unsigned char fraw[];
    const int tid = threadIdx.x;
    const FftSmem sm = fft_prologue<FFT_THREADS>(fraw, gf, gtw, tid);
    __syncthreads();
    const FftDev &f = *sm.f;
    float2 *A = sm.A, *B = A + f.bufsz;
    const int M = f.M, Mh = f.Mh, x = blockIdx.x, c = first + blockIdx.y;
    const float *g = grid + (size_t)c * pse_plane_stride(M) + (size_t)x * M * M;
    // two real rows per complex line (two-for-one): one conflict-free 8-byte shared store per pair of coalesced loads
    for (int idx = tid; idx < f.NP * M; idx += FFT_THREADS) {
        const int p = f.divM.div(idx), z = idx - p * M;
        const float a = g[(2 * p) * M + z], b = 2 * p + 1 < M ? g[(2 * p + 1) * M + z] : 0.f;
        A[p * f.Pz + z] = make_float2(a, b);
    }
    __syncthreads();
    fft_lines<false, FFT_THREADS>(A, B, f, 0, f.NP, f.divNP, f.Pz, 1, sm.tw, tid);
    // two-for-one separation: even line = (Z[k] + conj Z[M-k]) / 2, odd line = (Z[k] - conj Z[M-k]) / 2i
    for (int idx = tid; idx < f.NP * Mh; idx += FFT_THREADS) {
        const int p = f.divMh.div(idx), kz = idx - p * Mh;
        const float2 zk = A[p * f.Pz + kz], zm = A[p * f.Pz + (kz ? M - kz : 0)];
        B[(2 * p) * f.PK + kz] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
        if (2 * p + 1 < M) B[(2 * p + 1) * f.PK + kz] = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
    }
    __syncthreads();
    { float2 *t = A; A = B; B = t; }
    fft_lines<false, FFT_THREADS>(A, B, f, 0, Mh, f.divMh, 1, f.PK, sm.tw, tid);
    float4 *o = reinterpret_cast<float4 *>(spec + ((size_t)c * M + x) * M * f.Mhp);
    const float4 *a4 = reinterpret_cast<const float4 *>(A);
    for (int idx = tid; idx < (M * f.Mhp) >> 1; idx += FFT_THREADS) o[idx] = a4[idx];          // PK == Mhp: a straight copy
}

// ---- inverse: complex [M][Mhp] (ky, kz) -> real [M][M] (y, z) ----
__global__ void __launch_bounds__(FFT_THREADS, 2) fft_inv_plane_kernel(const float2 *__restrict__ spec, float *__restrict__ grid,
                                                                       const FftDev *__restrict__ gf, const float2 *__restrict__ gtw, int first) {
    extern __shared__ __align__(16) unsigned char fraw[];
    const int tid = threadIdx.x;
    const FftSmem sm = fft_prologue<FFT_THREADS>(fraw, gf, gtw, tid);
    __syncthreads();
    const FftDev &f = *sm.f;
    float2 *A = sm.A, *B = A + f.bufsz;
    const int M = f.M, Mh = f.Mh, x = blockIdx.x, c = first + blockIdx.y;
    const float4 *in = reinterpret_cast<const float4 *>(spec + ((size_t)c * M + x) * M * f.Mhp);
    float4 *a4 = reinterpret_cast<float4 *>(A);
    for (int idx = tid; idx < (M * f.Mhp) >> 1; idx += FFT_THREADS) a4[idx] = in[idx];
    __syncthreads();
    fft_lines<true, FFT_THREADS>(A, B, f, 0, Mh, f.divMh, 1, f.PK, sm.tw, tid);
    // two Hermitian lines a, b -> one complex line a + i b over all M frequencies
    for (int idx = tid; idx < f.NP * M; idx += FFT_THREADS) {
        const int p = f.divM.div(idx), k = idx - p * M;
        const bool lowk = k < Mh, has_b = 2 * p + 1 < M;
        const int ks = lowk ? k : M - k;
        float2 a = A[(2 * p) * f.PK + ks], b = has_b ? A[(2 * p + 1) * f.PK + ks] : make_float2(0.f, 0.f);
        if (!lowk) { a.y = -a.y; b.y = -b.y; }
        B[p * f.Pz + k] = make_float2(a.x - b.y, a.y + b.x);
    }
    __syncthreads();
    { float2 *t = A; A = B; B = t; }
    fft_lines<true, FFT_THREADS>(A, B, f, 0, f.NP, f.divNP, f.Pz, 1, sm.tw, tid);
    float *g = grid + (size_t)c * pse_plane_stride(M) + (size_t)x * M * M;
    for (int idx = tid; idx < f.NP * M; idx += FFT_THREADS) {
        const int p = f.divM.div(idx), z = idx - p * M;
        const float2 v = A[p * f.Pz + z];
        g[(2 * p) * M + z] = v.x;
        if (2 * p + 1 < M) g[(2 * p + 1) * M + z] = v.y;
    }
}

// rows (component c, kx) of the column (ky, kz0 .. kz0+7) between global memory and the [kx][slot][kzl] buffer,
// a float4 (two entries) per thread; float4s beyond the row pitch are zero-filled on load and skipped on store
template <bool LOAD>
__device__ __forceinline__ void xpass_copy(float2 *spec, float2 *A, int c0, int c1, int M, int Mhp, int ky, int kz0, int tid) {
    constexpr int QN = XCH / 2;                     // float4s per row chunk
    const int q = tid % QN, NL = 8 * XCH;
    const bool inside = kz0 + 2 * q < Mhp;
    const size_t plane = (size_t)M * M * Mhp;
    for (int c = c0; c < c1; ++c) {
        float2 *col = spec + c * plane + (size_t)ky * Mhp + kz0 + 2 * q;
#pragma unroll 2
        for (int kx = tid / QN; kx < M; kx += XT / QN) {
            float4 *s = reinterpret_cast<float4 *>(A + kx * NL + c * XCH + 2 * q);
            float4 *gp = reinterpret_cast<float4 *>(col + (size_t)kx * M * Mhp);
            if (LOAD) *s = inside ? *gp : make_float4(0.f, 0.f, 0.f, 0.f);
            else if (inside) *gp = *s;
        }
    }
}

// ---- x pass fused with the k-space operator: forward along x, P^H B P at every mode, inverse along x ----
// Shared layout [kx][slot][kzl]: slot = absolute component 0..7 (F/U in 0-2, S/E in 3-7), kzl < XCH fastest, so the
// line index (slot, kzl) is contiguous and the component stride is XCH: write_outputs / scale_point apply unchanged.
__global__ void __launch_bounds__(XT, 4) fft_x_scale_kernel(float2 *__restrict__ spec, ScaleParams sp, const FftDev *__restrict__ gf,
                                                                     const float2 *__restrict__ gtw, FastDiv xdiv_in, FastDiv xdiv_out) {
    extern __shared__ __align__(16) unsigned char fraw[];
    const int tid = threadIdx.x;
    const FftSmem sm = fft_prologue<XT>(fraw, gf, gtw, tid);
    const int M = gf->M, Mh = gf->Mh, Mhp = gf->Mhp, NL = 8 * XCH;
    float2 *A = sm.A, *B = A + (size_t)M * NL;
    const int ky = blockIdx.x, kz0 = blockIdx.y * XCH;
    const int in0 = (sp.mode & PSE_IN_F) ? 0 : 3, in1 = (sp.mode & PSE_IN_S) ? 8 : 3;
    const int out0 = (sp.mode & PSE_OUT_U) ? 0 : 3, out1 = (sp.mode & PSE_OUT_E) ? 8 : 3;
    xpass_copy<true>(spec, A, in0, in1, M, Mhp, ky, kz0, tid);
    __syncthreads();
    const FftDev &f = *sm.f;
    fft_lines<false, XT>(A, B, f, in0 * XCH, (in1 - in0) * XCH, xdiv_in, 1, NL, sm.tw, tid);
    for (int idx = tid; idx < M * XCH; idx += XT) {
        const int kzl = idx & (XCH - 1), kx = idx / XCH;
        if (kz0 + kzl < Mh) scale_point(sp, kx, ky, kz0 + kzl, A, XCH, (size_t)kx * NL + kzl, A, XCH, (size_t)kx * NL + kzl);
        else {
            for (int c = out0; c < out1; ++c) A[kx * NL + c * XCH + kzl] = make_float2(0.f, 0.f);
        }
    }
    __syncthreads();
    fft_lines<true, XT>(A, B, f, out0 * XCH, (out1 - out0) * XCH, xdiv_out, 1, NL, sm.tw, tid);
    xpass_copy<false>(spec, A, out0, out1, M, Mhp, ky, kz0, tid);
}

// inverse x pass alone (Brownian displacement: the spectrum is written by scale_brownian_kernel)
__global__ void __launch_bounds__(XT, 4) fft_x_inv_kernel(float2 *__restrict__ spec, const FftDev *__restrict__ gf,
                                                                   const float2 *__restrict__ gtw, FastDiv xdiv_out) {
    extern __shared__ __align__(16) unsigned char fraw[];
    const int tid = threadIdx.x;
    const FftSmem sm = fft_prologue<XT>(fraw, gf, gtw, tid);
    const int M = gf->M, Mhp = gf->Mhp, NL = 8 * XCH;
    float2 *A = sm.A, *B = A + (size_t)M * NL;
    const int ky = blockIdx.x, kz0 = blockIdx.y * XCH;
    xpass_copy<true>(spec, A, 0, 8, M, Mhp, ky, kz0, tid);
    __syncthreads();
    fft_lines<true, XT>(A, B, *sm.f, 0, 8 * XCH, xdiv_out, 1, NL, sm.tw, tid);
    xpass_copy<false>(spec, A, 0, 8, M, Mhp, ky, kz0, tid);
}

// fewest stages with radices the kernels implement (depth-first; M <= a few hundred)
bool factor_rec(int m, int depth, int maxdepth, int *cur, int *best, int &nbest) {
    static const int cand[] = {16, 12, 10, 9, 8, 6, 5, 4, 3, 2};
    if (m == 1) { if (depth < nbest) { nbest = depth; for (int i = 0; i < depth; ++i) best[i] = cur[i]; } return true; }
    if (depth + 1 >= nbest || depth >= maxdepth) return false;
    bool ok = false;
    for (int r : cand) if (m % r == 0) { cur[depth] = r; ok |= factor_rec(m / r, depth + 1, maxdepth, cur, best, nbest); }
    return ok;
}
bool factorise(int M, int *radix, int &n) {
    int cur[8], best[8], nbest = FFT_MAXSTAGE + 1;
    if (M < 2 || !factor_rec(M, 0, FFT_MAXSTAGE, cur, best, nbest)) return false;
    n = nbest;
    for (int i = 0; i < n; ++i) radix[i] = best[i];
    return true;
}

bool make_fft(int M, FftDev &f) {
    int radix[8], n = 0;
    if (!factorise(M, radix, n)) return false;
    f.M = M; f.Mh = M / 2 + 1; f.Mhp = (f.Mh + 3) & ~3; f.nstage = n;
    for (int i = 0, ns = 1; i < n; ++i) {
        f.st[i].R = radix[i]; f.st[i].Ns = ns; f.st[i].nb = M / radix[i]; f.st[i].tstep = M / (ns * radix[i]); f.st[i].ns_div = make_div(ns);
        ns *= radix[i];
    }
    f.NP = (M + 1) / 2;
    f.Pz = M | 1;                                 // odd pitch: lanes over lines hit distinct banks
    f.PK = f.Mhp;
    f.bufsz = (std::max(f.NP * f.Pz, M * f.PK) + 1) & ~1;
    f.divM = make_div(M); f.divMh = make_div(f.Mh); f.divNP = make_div(f.NP); f.divMq = make_div(std::max(1, M / 4));
    return true;
}

}  // namespace

// Decides whether the own FFT serves this grid (opt-in: PSE_FFT=own), sets the spectrum pitch and uploads plan record
// and twiddles.
pse_status pse_fft_init(pse_ctx *c) {
    c->own_fft = false;
    c->Mhp = c->Mh;
    // Measured on B200 at 100^3, five planes: forward planes 32-34 us, x pass with the operator 41-44 us, inverse planes
    // 33-34 us against cuFFT's 40 + 15 (scale_kernel) + 41 us: the fusion saves four passes over the spectrum, but
    // the kernels are bound by instruction issue and barriers (ncu: issue active 45-55 %), not by memory, so the saving does
    // not show.  cuFFT therefore stays the default and PSE_FFT=own selects this path (parity-tested either way).
    const char *e = getenv("PSE_FFT");
    if (!e || std::string(e) != "own") return PSE_OK;
    FftDev f;
    if (c->M < 8 || c->M > 1024 || !make_fft(c->M, f)) return PSE_OK;
    int dev = 0, max_smem = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t plane = fft_prologue_bytes(c->M) + 2 * (size_t)f.bufsz * sizeof(float2);
    const size_t xpass = fft_prologue_bytes(c->M) + 2 * (size_t)c->M * 8 * XCH * sizeof(float2);
    if (plane > (size_t)max_smem || xpass > (size_t)max_smem) return PSE_OK;
    std::vector<float> tw(2 * (size_t)c->M);
    for (int i = 0; i < c->M; ++i) { const double t = -2.0 * M_PI * i / c->M; tw[2 * i] = (float)std::cos(t); tw[2 * i + 1] = (float)std::sin(t); }
    CUDA_TRY(c, cudaMalloc(&c->d_fft_tw, tw.size() * sizeof(float)));
    CUDA_TRY(c, cudaMemcpy(c->d_fft_tw, tw.data(), tw.size() * sizeof(float), cudaMemcpyHostToDevice));
    CUDA_TRY(c, cudaMalloc(&c->d_fft_dev, sizeof(FftDev)));
    CUDA_TRY(c, cudaMemcpy(c->d_fft_dev, &f, sizeof(FftDev), cudaMemcpyHostToDevice));
    CUDA_TRY(c, cudaFuncSetAttribute(fft_fwd_plane_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plane));
    CUDA_TRY(c, cudaFuncSetAttribute(fft_inv_plane_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plane));
    CUDA_TRY(c, cudaFuncSetAttribute(fft_x_scale_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xpass));
    CUDA_TRY(c, cudaFuncSetAttribute(fft_x_inv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xpass));
    c->fft_smem_plane = plane; c->fft_smem_x = xpass;
    c->Mhp = f.Mhp;
    c->own_fft = true;
    return PSE_OK;
}

// planes [first, first+ncomp) of d_grid -> d_spec (y and z transformed; x still in real space)
pse_status pse_fft_forward_planes(pse_ctx *c, int first, int ncomp) {
    fft_fwd_plane_kernel<<<dim3(c->M, ncomp), FFT_THREADS, c->fft_smem_plane, c->stream>>>(
        c->d_grid, reinterpret_cast<float2 *>(c->d_spec), static_cast<const FftDev *>(c->d_fft_dev), reinterpret_cast<const float2 *>(c->d_fft_tw), first);
    KERNEL_CHECK(c);
    return PSE_OK;
}

// x transform, k-space operator, inverse x transform, in place in d_spec
pse_status pse_fft_x_scale(pse_ctx *c, int mode) {
    const int nin = (mode & PSE_IN_F ? 3 : 0) + (mode & PSE_IN_S ? 5 : 0), nout = (mode & PSE_OUT_U ? 3 : 0) + (mode & PSE_OUT_E ? 5 : 0);
    fft_x_scale_kernel<<<dim3(c->M, (c->Mh + XCH - 1) / XCH), XT, c->fft_smem_x, c->stream>>>(
        reinterpret_cast<float2 *>(c->d_spec), make_scale_params(c, mode), static_cast<const FftDev *>(c->d_fft_dev),
        reinterpret_cast<const float2 *>(c->d_fft_tw), make_div(nin * XCH), make_div(nout * XCH));
    KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_fft_x_inverse(pse_ctx *c) {
    fft_x_inv_kernel<<<dim3(c->M, (c->Mh + XCH - 1) / XCH), XT, c->fft_smem_x, c->stream>>>(
        reinterpret_cast<float2 *>(c->d_spec), static_cast<const FftDev *>(c->d_fft_dev), reinterpret_cast<const float2 *>(c->d_fft_tw), make_div(8 * XCH));
    KERNEL_CHECK(c);
    return PSE_OK;
}

pse_status pse_fft_inverse_planes(pse_ctx *c, int first, int ncomp) {
    fft_inv_plane_kernel<<<dim3(c->M, ncomp), FFT_THREADS, c->fft_smem_plane, c->stream>>>(
        reinterpret_cast<const float2 *>(c->d_spec), c->d_grid, static_cast<const FftDev *>(c->d_fft_dev), reinterpret_cast<const float2 *>(c->d_fft_tw), first);
    KERNEL_CHECK(c);
    return PSE_OK;
}

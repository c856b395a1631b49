// pse_hard_sphere_forces_noalloc: the Heyes-Melrose overlap force (reading R12, include/pse.h) for callers that
// cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).  No context, no
// allocation: the linked-cell scratch that pse_neighbors keeps in context-owned cudaMalloc buffers lives here in ONE
// file-scope __device__ array of fixed size, which every GPU that loads the library holds until the process exits.
//
//   scratch layout   int head[PSE_NOALLOC_MAX_CELLS]   first particle of every cell, -1 = empty (cleared by every call)
//                    int next[PSE_NOALLOC_MAX_N]       next particle of the same cell, -1 = end (written for i < N by every call)
//
// In host code the array's NAME is a host-side stand-in, not a device address; the address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current (scratch_of_current_device below).
// Every call shares the array: two calls that overlap on the GPU (different streams, or different host threads without
// ordering) race on it.  Calls on one stream are ordered and safe.
//
// Arithmetic per pair is that of hs_forces in neighbors.cu (wrapped coordinates, minimum image, fp32); the sum over the
// overlapping partners of a particle runs over the 27 (fewer in a box under 3 cells) neighbour cells in a fixed order and,
// inside a cell, in ascending particle index, so the result does not depend on the order in which the atomics linked the cells.
#include <cuda_runtime.h>

#include <climits>
#include <cmath>
#include <cstdio>
#include <mutex>

#include "pse.h"

namespace {

constexpr int MAX_N = PSE_NOALLOC_MAX_N;
constexpr int MAX_NC = 64;                                    // cells per dimension
constexpr int MAX_CELLS = MAX_NC * MAX_NC * MAX_NC;
constexpr int ORDERED_MAX = 32;                               // cells fuller than this are summed in list order (see hs_cells_kernel)
constexpr int MAX_DEVICES = 64;
constexpr size_t SCRATCH_BYTES = ((size_t)MAX_CELLS + (size_t)MAX_N) * sizeof(int);
static_assert(SCRATCH_BYTES == PSE_NOALLOC_SCRATCH_BYTES, "include/pse.h states the size of the static scratch");

static __device__ __align__(256) unsigned char g_noalloc_scratch[SCRATCH_BYTES];

std::mutex g_mu;
void *g_scratch_dev[MAX_DEVICES];                             // device address of g_noalloc_scratch on every device asked so far

void say(char *h_err, size_t cap, const char *msg, double v = 0, double w = 0) {
    if (h_err && cap) snprintf(h_err, cap, msg, v, w);
}

// the device address of the scratch on the CURRENT device (looked up once per device)
cudaError_t scratch_of_current_device(void **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_dev[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_dev[dev] = p;
    }
    *out = g_scratch_dev[dev];
    return cudaSuccess;
}

__device__ __forceinline__ float wrap_coord(float x, float L, float invL) {
    float w = __fsub_rn(x, __fmul_rn(L, floorf(__fmul_rn(x, invL))));
    return (w >= L || w < 0.f) ? 0.f : w;
}
__device__ __forceinline__ float min_image(float d, float L, float invL) {
    return __fsub_rn(d, __fmul_rn(L, rintf(__fmul_rn(d, invL))));
}
__device__ __forceinline__ int cell_coord(float w, float cell_inv, int nc) { return min(nc - 1, (int)(w * cell_inv)); }

// next[i] = previous head of i's cell, head = i
__global__ void link_cells_kernel(const float4 *__restrict__ pos, int N, float L, float invL, int nc, float cell_inv,
                                  int *__restrict__ head, int *__restrict__ next) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 p = pos[i];
    const int cx = cell_coord(wrap_coord(p.x, L, invL), cell_inv, nc), cy = cell_coord(wrap_coord(p.y, L, invL), cell_inv, nc),
              cz = cell_coord(wrap_coord(p.z, L, invL), cell_inv, nc);
    next[i] = atomicExch(&head[(cx * nc + cy) * nc + cz], i);
}

// F_i = sum_{j != i, r_ij < 2a} coef (2a - r_ij)/r_ij (x_i - x_j)_min-image, thread per particle
__global__ void hs_cells_kernel(const float4 *__restrict__ pos, int N, float L, float invL, int nc, float cell_inv,
                                const int *__restrict__ head, const int *__restrict__ next, float two_a, float coef, float *__restrict__ F) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i];
    p.x = wrap_coord(p.x, L, invL); p.y = wrap_coord(p.y, L, invL); p.z = wrap_coord(p.z, L, invL);
    const int cx = cell_coord(p.x, cell_inv, nc), cy = cell_coord(p.y, cell_inv, nc), cz = cell_coord(p.z, cell_inv, nc);
    const int span = min(nc, 3);                              // distinct cells among {c-1, c, c+1} mod nc
    float fx = 0.f, fy = 0.f, fz = 0.f;
    auto pair = [&](int j) {
        if (j == i) return;
        float4 q = pos[j];
        q.x = wrap_coord(q.x, L, invL); q.y = wrap_coord(q.y, L, invL); q.z = wrap_coord(q.z, L, invL);
        const float dx = min_image(p.x - q.x, L, invL), dy = min_image(p.y - q.y, L, invL), dz = min_image(p.z - q.z, L, invL);
        const float r2 = dx * dx + dy * dy + dz * dz;
        if (r2 < two_a * two_a && r2 > 0.f) {
            const float r = sqrtf(r2), g = coef * (two_a - r) / r;
            fx += g * dx; fy += g * dy; fz += g * dz;
        }
    };
    for (int ox = 0; ox < span; ++ox)
        for (int oy = 0; oy < span; ++oy)
            for (int oz = 0; oz < span; ++oz) {
                const int c = (((cx - 1 + ox + nc) % nc) * nc + (cy - 1 + oy + nc) % nc) * nc + (cz - 1 + oz + nc) % nc;
                int n = 0;
                for (int j = head[c]; j >= 0 && n <= ORDERED_MAX; j = next[j]) ++n;
                if (n <= ORDERED_MAX) {                       // ascending index: repeated search for the smallest index above the last
                    for (int last = -1;;) {
                        int best = INT_MAX;
                        for (int j = head[c]; j >= 0; j = next[j])
                            if (j > last && j < best) best = j;
                        if (best == INT_MAX) break;
                        pair(best);
                        last = best;
                    }
                } else {                                      // a crowded cell (far beyond any hard-sphere packing): list order
                    for (int j = head[c]; j >= 0; j = next[j]) pair(j);
                }
            }
    F[3 * (size_t)i] = fx; F[3 * (size_t)i + 1] = fy; F[3 * (size_t)i + 2] = fz;
}

}  // namespace

extern "C" pse_status pse_hard_sphere_forces_noalloc(int N, double L, double a, double eta, double dt, const float *d_pos, float *d_F,
                                                     void *cuda_stream, char *h_err, size_t h_err_cap) {
    if (h_err && h_err_cap) h_err[0] = '\0';
    if (N <= 0 || !(L > 0) || !(a > 0) || !(eta > 0) || !(dt > 0) || !d_pos || !d_F) {
        say(h_err, h_err_cap, "pse_hard_sphere_forces_noalloc: non-positive or missing argument");
        return PSE_EINVAL;
    }
    if (N > MAX_N) {
        say(h_err, h_err_cap, "pse_hard_sphere_forces_noalloc: N = %.0f exceeds the static scratch (PSE_NOALLOC_MAX_N = %.0f); "
                              "use pse_neighbors + pse_hard_sphere_forces", (double)N, (double)MAX_N);
        return PSE_EOVERFLOW;
    }
    if (4.0 * a > L) {
        say(h_err, h_err_cap, "pse_hard_sphere_forces_noalloc: contact distance 2a = %g > L/2 = %g (minimum image)", 2.0 * a, 0.5 * L);
        return PSE_EINVAL;
    }
    void *scratch = nullptr;
    cudaError_t e = scratch_of_current_device(&scratch);
    if (e != cudaSuccess) {
        if (h_err && h_err_cap) snprintf(h_err, h_err_cap, "pse_hard_sphere_forces_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return PSE_ECUDA;
    }
    // cell edge L/nc >= 2a (1 + 1e-4): the fp32 cell coordinate is off by at most ~64 * 2^-23 cells, so partners closer than 2a
    // are never two cells apart
    int nc = (int)std::floor(L / (2.0 * a) * (1.0 - 1e-4));
    nc = nc < 1 ? 1 : (nc > MAX_NC ? MAX_NC : nc);
    const size_t ncell = (size_t)nc * nc * nc;
    int *head = static_cast<int *>(scratch), *next = head + MAX_CELLS;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const float Lf = (float)L, invL = 1.0f / Lf, cell_inv = (float)(nc / L);
    const int T = 256, nb = (N + T - 1) / T;
    e = cudaMemsetAsync(head, 0xFF, ncell * sizeof(int), s);  // what must start clean: every head = -1
    if (e == cudaSuccess) {
        link_cells_kernel<<<nb, T, 0, s>>>(reinterpret_cast<const float4 *>(d_pos), N, Lf, invL, nc, cell_inv, head, next);
        hs_cells_kernel<<<nb, T, 0, s>>>(reinterpret_cast<const float4 *>(d_pos), N, Lf, invL, nc, cell_inv, head, next, (float)(2 * a),
                                         (float)(3.0 * M_PI * eta * a / dt), d_F);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (h_err && h_err_cap) snprintf(h_err, h_err_cap, "pse_hard_sphere_forces_noalloc: %s", cudaGetErrorString(e));
        return PSE_ECUDA;
    }
    return PSE_OK;
}

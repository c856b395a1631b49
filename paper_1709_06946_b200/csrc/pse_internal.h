// Internal declarations of libpse (not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>
#include "pse.h"

#define PSE_NTAB 2048          // nodes of the real-space table (8 floats each -> 64 KB, staged in shared memory)
#define PSE_TILE 8             // spread / interpolate tile edge in grid points
#define PSE_MAXP 16
#define PSE_MAX_KRYLOV 50

// which components a product carries: inputs F (3) and/or S (5), outputs U (3) and/or E (5).  Inside GMRES the operator
// is S -> E only, so 5 + 5 grids are spread / transformed / interpolated instead of 8 + 8.
enum { PSE_IN_F = 1, PSE_IN_S = 2, PSE_OUT_U = 4, PSE_OUT_E = 8, PSE_MODE_ALL = 15 };

#define PSE_GRAPH_MAX_N (1 << 30)  // pse_step replays captured CUDA graphs up to this many particles (all sizes: it pays everywhere measured)

struct Timer { cudaEvent_t a, b; int phase; };

// Deformed periodic lattice (NEXT-4; Eqs. 56, 58): lattice vectors = columns of L A with
// A = [[a11, a12, 0], [0, a22, 0], [0, 0, 1]], det A = 1 (simple shear: a12 = gamma; planar extension: a11 = 1/a22 = epsilon).
// Inside the library positions are LATTICE coordinates s = A^-1 x wrapped into [0, L)^3, so binning, spreading and interpolation
// are those of the cube; physical separations r = A d (d = minimum image of s_a - s_b) and wave vectors k = (2 pi/L) A^-T n
// appear only where distances and the Green's function are evaluated (reading R22).  i** = entries of A^-1.
struct Lat { float a11, a12, a22, i11, i12, i22; };
// cells of the neighbour search per lattice direction: edge L/n_i >= r_cut * (norm of row i of A^-1), so a deformed cell is not searched
// with cubes sized for its worst direction
struct Cells { int x, y, z; };

// everything baked into the captured graph of a step
struct StepGraphKey {
    const void *pos, *noise_real, *noise_wave; double dt; int mL, mG, n_bonds; size_t nbr_cap; int ncx, ncy, ncz; bool deformed;
    bool operator==(const StepGraphKey &o) const {
        return pos == o.pos && noise_real == o.noise_real && noise_wave == o.noise_wave && dt == o.dt && mL == o.mL && mG == o.mG &&
               n_bonds == o.n_bonds && nbr_cap == o.nbr_cap && ncx == o.ncx && ncy == o.ncy && ncz == o.ncz && deformed == o.deformed;
    }
};

// Everything the tiled interpolation needs about one grid: the product grid (M, P) or the finer grid of the Brownian pass.
struct InterpSet {
    int M = 0, P = 0, PP = 0, nt = 0, ntile = 0;
    float *grid = nullptr;                   // [8][pse_plane_stride(M)]
    int *tile_start = nullptr, *tile_list = nullptr;     // bins of the particles by the tile of their support base
    int *pbase = nullptr; float *pw = nullptr;           // per-particle window data in tile order
    CUtensorMap tmap;                        // TMA descriptor of grid as [8][M][M][M] with the (T+P-1)^3 box
    bool tma_ok = false;
};

struct pse_ctx {
    // ---- parameters (pse_create) ----
    int N = 0, M = 0, P = 0;
    double L = 0, a = 0, eta = 0, kT = 0, xi = 0, rcut = 0, tol = 0;
    double h = 0, eta_g = 0;                 // grid spacing, Gaussian shape parameter
    double lat_a11 = 1, lat_a12 = 0, lat_a22 = 1;   // the lattice deformation A (pse_set_lattice); identity = the cubic box
    bool deformed = false;
    Lat *d_lat = nullptr;                    // A and A^-1 in device memory: what the kernels read, so that a captured step outlives a change of strain
    int win_kind = 1;                        // 0 = Gaussian (paper), 1 = exponential-of-semicircle window
    double win_a = 0, win_b = 0;             // window parameters handed to the kernels (see win_arg in wavespace.cu)
    float *d_dec = nullptr;                  // [M] inverse 1-D window transform per FFT index
    // ---- finer grid of the Brownian wave pass (the field sqrt(B) W decays only like exp(-k^2/8 xi^2), so the modes
    //      next to the Nyquist frequency of the product grid, which a P-point window cannot interpolate, still carry weight;
    //      the same modes are therefore evaluated on a grid Mb > M: zero-padded spectrum, own C2R plan, generic interpolation) ----
    int Mb = 0, Mbh = 0, Pb = 0;             // Pb = P + 1 support points per dimension
    double win_a_b = 0, win_b_b = 0;         // window parameters for Pb
    float *d_dec_b = nullptr;                // [Mb]
    float *d_grid_b = nullptr;               // [8][Mb^3]
    cufftComplex *d_spec_b = nullptr;        // [8][Mb][Mb][Mbh]
    cufftHandle plan_c2r_b = 0; bool have_plan_b = false;
    cudaStream_t stream = nullptr;
    int device = 0, nsm = 0;                 // device the context lives on (recorded at pse_create), its SM count
    int coop_cap = 0;                        // largest cooperative grid of the Krylov step kernels on that device
    cudaStream_t stream2 = nullptr;          // pse_step_host uploads the noise here while the step starts on `stream`
    cudaStream_t stream_cap = nullptr;       // pse_step's graph is captured here (the caller's stream may be the legacy default stream)
    cudaEvent_t ev_fork = nullptr, ev_noise = nullptr, ev_noise_r = nullptr;
    bool noise_r_pending = false;            // pse_step_host: the real-space noise upload on stream2 has not been waited for yet
    bool noise_pending = false;              // pse_step_host: the wave-noise upload on stream2 has not been waited for yet
    std::string err;
    long long launches = 0;
    // ---- real-space table ----
    float *d_table = nullptr;                // [PSE_NTAB][8]
    double tab_dr = 0;
    // ---- cell list / neighbour list (all in cell-sorted numbering unless noted) ----
    Cells nc = {0, 0, 0};                    // cells per lattice direction
    int ncell = 0, ncell_cap = 0;            // their product; what the cell arrays were allocated for (the cube's count)
    bool have_nbrs = false;
    float4 *d_pos = nullptr;                 // [N] wrapped positions, sorted
    int *d_order = nullptr;                  // [N] sorted -> original
    int *d_order_tmp = nullptr, *d_tile_tmp = nullptr;   // [N] unsorted scatter targets
    int *d_cell_of = nullptr;                // [N] cell of original particle
    int *d_bins = nullptr; size_t bins_n = 0;   // one block cleared by a single memset: cell_count | cell_fill | tile_count | tile_fill | half_cursor
    int *d_cell_count = nullptr, *d_cell_start = nullptr, *d_cell_fill = nullptr;   // [ncell+1]; count and fill point into d_bins
    int *d_nbr_count = nullptr;              // [N]
    unsigned long long *d_nbr_off = nullptr; // [N+1]
    int *d_nbr_idx = nullptr; size_t nbr_cap = 0, nbr_total = 0;
    unsigned long long *d_nbr_ctl = nullptr, *h_nbr_ctl = nullptr;   // {allocation cursor, fallback flag}; pinned mirror, two slots of two
    int nbr_slot = 0, nbr_last = 0;          // slot of h_nbr_ctl the next build reports into / the last one did
    cudaEvent_t ev_nbr = nullptr;            // recorded behind the build's read-back
    bool nbr_pending = false;                // the last build's size / flags have not been examined yet (pse_neighbors_settle)
    bool nbr_two_pass = false;               // a cell once exceeded the mask store: this context takes the two-pass path
    // ---- FFT-grid tile bins ----
    int nt = 0, ntile = 0, Mh = 0;           // tiles per dimension, total, M/2+1
    int *d_tile_count = nullptr, *d_tile_start = nullptr, *d_tile_fill = nullptr;   // [ntile+1]; count and fill point into d_bins
    int *d_tile_of = nullptr;                // [N] tile of the particle's support base, original numbering
    int *d_tile_list = nullptr;              // [N] sorted-particle indices grouped by tile
    // ---- per-particle window data, computed once per pse_neighbors and shared by every spread / interpolation of that
    //      configuration (a step runs ~25 of them on two configurations) ----
    int *d_pbase = nullptr;                  // [N] wrapped support base, packed bx | by << 10 | bz << 20; TILE ORDER: entry i is particle d_tile_list[i]
    float *d_pw = nullptr;                   // [N][3][PP] (tile order) window values at the P support points per dimension, PP = P rounded up to 4
    int PP = 0;
    // particles that reach each half tile (4 x 8 x 8 grid points, one warp of the spread kernel): CSR, built in pse_neighbors
    int *d_half_cursor = nullptr;            // allocation cursor of d_half_list, inside d_bins (cleared by its memset)
    int *d_half_start = nullptr, *d_half_count = nullptr, *d_half_list = nullptr;   // [2 ntile] segment start / length; entries = tile-order indices
    size_t half_cap = 0;
    // ---- grids ----
    float *d_grid = nullptr;                 // [8][M][M][M]
    cufftComplex *d_spec = nullptr;          // [8][M][M][Mh]
    cufftHandle plan_r2c[3] = {0, 0, 0}, plan_c2r[3] = {0, 0, 0};   // [0] all 8 grids, [1] planes 0-2 (F / U), [2] planes 3-7 (S / E)
    void *d_fft_work = nullptr; int nplans = 0;
    InterpSet iset, iset_b;                  // interpolation views of the product grid and of the Brownian pass's finer grid
    int *d_tile_of_b = nullptr, *d_tile_tmp_b = nullptr, *d_tile_cnt_b = nullptr;   // binning scratch of the finer grid ([N], [N], [2 (ntile_b + 1)])
    bool fine_bins_valid = false;            // iset_b's bins and window data belong to the current positions
    // ---- packed per-particle vectors, sorted numbering: [N][8] = (x,y,z,e1..e5) ----
    float *d_in = nullptr, *d_out = nullptr, *d_tmp = nullptr, *d_tmp2 = nullptr;
    float *d_krylov = nullptr;  int krylov_cap = 0;      // [krylov_cap][N][8]
    float *d_zu = nullptr;                               // [PSE_MAX_KRYLOV][N][8] full outputs M[0;v_j] (GMRES)
    double *d_scal = nullptr;                // device scalars (dots, norms)
    double *h_scal = nullptr;                // pinned mirror
    double *h_scal_l = nullptr;              // pinned mirror of the Lanczos scalars of a fixed-count solve (pse_step's optimistic path)
    int lanczos_budget = 0, gmres_budget = 0;   // iteration counts the last completed step needed; 0 = not known yet
    float4 *d_xk = nullptr;                  // [N] copy of x_k while an optimistic step is in flight
    cudaGraphExec_t step_graph[3] = {nullptr, nullptr, nullptr};   // the fixed-count step as three graphs: [build], [Lanczos], [wave sample ... update]
    StepGraphKey graph_key = {};
    int graph_slot0 = 0, graph_slot1 = 0; long long graph_launches = 0; bool graph_failed = false; int graph_recaptures = 0;
    float *d_coef = nullptr;                 // small coefficient vector upload
    int last_lanczos_iters = 0, last_gmres_iters = 0;   // iteration counts of the previous solves (when to start reading back)
    int lanczos_repeats = 0, gmres_repeats = 0;         // how many solves in a row ended with that same count
    unsigned long long *d_scan_tmp = nullptr; size_t scan_tmp_n = 0;
    float4 *d_posw = nullptr;                // [N] wrapped positions, original numbering
    float *d_vecA = nullptr, *d_vecB = nullptr, *d_vecC = nullptr, *d_vecD = nullptr;   // [N][8] scratch for pse_step
    // ---- full couplet (torque in, angular velocity out; couplet.cu), allocated by the first call that needs them ----
    float *d_rot_table = nullptr;            // [PSE_NTAB][4] = (T/2, Z0/6, Z2/4, 0)/(6 pi eta a) at the nodes of d_table
    cufftComplex *d_spec_rot = nullptr;      // [3][M][M][Mh] spectrum of the torque planes in, of the angular-velocity planes out
    float *d_rot_in = nullptr, *d_rot_out = nullptr, *d_rot_tmp = nullptr;   // [N][8] packed: (Lx,Ly,Lz,0..), (Ox,Oy,Oz,0..), scratch
    float *d_rot_w = nullptr, *d_rot_y = nullptr, *d_rot_u = nullptr;        // [2][N][8] each: 11-component Lanczos input, result, work vector
    cufftComplex *d_spec_rot_b = nullptr;    // [3][Mb][Mb][Mbh] angular-velocity spectra of the Brownian pass (finer grid)
    cufftHandle plan_c2r_rot_b = 0; bool have_plan_rot_b = false;
    // ---- bonds of the equilibrium test potential U = k |r - r0|, original numbering ----
    int2 *d_bonds = nullptr; int n_bonds = 0; double bond_k = 0, bond_r0 = 0;
    // ---- staging for the host-buffer entry points ----
    float *d_stage_pos = nullptr, *d_stage_a = nullptr, *d_stage_b = nullptr, *d_stage_noise = nullptr;
    // ---- profiling ----
    bool profiling = false;
    std::vector<Timer> timers;
    float acc_ms[PSE_T_COUNT] = {0};
    int acc_n[PSE_T_COUNT] = {0};
};

#define CUDA_TRY(ctx, expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { \
    (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e_); return PSE_ECUDA; } } while (0)
#define CUFFT_TRY(ctx, expr) do { cufftResult r_ = (expr); if (r_ != CUFFT_SUCCESS) { \
    (ctx)->err = std::string(#expr) + ": cufft error " + std::to_string((int)r_); return PSE_ECUFFT; } } while (0)
#define PSE_TRY(expr) do { pse_status s_ = (expr); if (s_ != PSE_OK) return s_; } while (0)
#define KERNEL_CHECK(ctx) do { (ctx)->launches++; CUDA_TRY(ctx, cudaGetLastError()); } while (0)

struct ScopedPhase {
    pse_ctx *c; int idx = -1;
    ScopedPhase(pse_ctx *ctx, int phase) : c(ctx) {
        if (!c->profiling || phase < 0) return;
        Timer t; t.phase = phase;
        cudaEventCreate(&t.a); cudaEventCreate(&t.b);
        cudaEventRecord(t.a, c->stream);
        c->timers.push_back(t); idx = (int)c->timers.size() - 1;
    }
    ~ScopedPhase() { if (idx >= 0) cudaEventRecord(c->timers[idx].b, c->stream); }
};

// Distance in floats between two of the 8 real grids: M^3 rounded up to a multiple of 4, so that every plane starts
// 16-byte aligned (cuFFT rejects a real batch pointer that is only 4-byte aligned: odd M, odd first plane).
#ifdef __CUDACC__
__host__ __device__
#endif
inline size_t pse_plane_stride(int M) { return ((size_t)M * M * M + 3) & ~(size_t)3; }

#ifdef __CUDACC__
// support base (unwrapped, may be negative) of grid coordinate g = x/h   (reading R5)
__device__ __forceinline__ int pse_support_base(float g, int P) {
    return (P & 1) ? (int)rintf(g) - (P - 1) / 2 : (int)floorf(g) - P / 2 + 1;
}
// periodic index for arguments in [-M, 2M) (support bases and offsets never leave that range since P <= M): no division
__device__ __forceinline__ int pse_pmod(int i, int M) { i += i < 0 ? M : 0; return i >= M ? i - M : i; }
// spread / interpolate tile (edge PSE_TILE grid points) that holds the support base of a wrapped position
__device__ __forceinline__ int pse_tile_of(float4 p, float inv_h, int M, int P, int nt) {
    const int tx = pse_pmod(pse_support_base(p.x * inv_h, P), M) / PSE_TILE, ty = pse_pmod(pse_support_base(p.y * inv_h, P), M) / PSE_TILE,
              tz = pse_pmod(pse_support_base(p.z * inv_h, P), M) / PSE_TILE;
    return (tx * nt + ty) * nt + tz;
}
// Warp reduction of 8 per-lane partial sums with 9 shuffles instead of 40: each step halves the number of values a
// lane carries.  On return the lanes with (lane & 3) == 0 hold the full sum of component
// comp = 4*bit4(lane) + 2*bit3(lane) + bit2(lane).
__device__ __forceinline__ float warp_reduce8(const float (&a)[8], int lane, int &comp) {
    const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
    float r4[4], r2[2];
#pragma unroll
    for (int c = 0; c < 4; ++c) r4[c] = (h16 ? a[c + 4] : a[c]) + __shfl_xor_sync(0xffffffffu, h16 ? a[c] : a[c + 4], 16);
#pragma unroll
    for (int c = 0; c < 2; ++c) r2[c] = (h8 ? r4[c + 2] : r4[c]) + __shfl_xor_sync(0xffffffffu, h8 ? r4[c] : r4[c + 2], 8);
    float r = (h4 ? r2[1] : r2[0]) + __shfl_xor_sync(0xffffffffu, h4 ? r2[0] : r2[1], 4);
    r += __shfl_xor_sync(0xffffffffu, r, 2);
    r += __shfl_xor_sync(0xffffffffu, r, 1);
    comp = (h16 ? 4 : 0) + (h8 ? 2 : 0) + (h4 ? 1 : 0);
    return r;
}
#endif

inline Lat pse_lat(const pse_ctx *c) {
    Lat l;
    l.a11 = (float)c->lat_a11; l.a12 = (float)c->lat_a12; l.a22 = (float)c->lat_a22;
    l.i11 = (float)(1.0 / c->lat_a11); l.i12 = (float)(-c->lat_a12 / (c->lat_a11 * c->lat_a22)); l.i22 = (float)(1.0 / c->lat_a22);
    return l;
}

// api.cu
int pse_choose_grid(int mmin);
// tables.cu
void pse_build_table(double a, double eta, double xi, double rcut, int ntab, std::vector<float> &tab, double *dr);
void pse_window_table(int kind, int P, double wa, double wb, int M, std::vector<float> &dec);
double pse_es_beta(int P);
// neighbors.cu
pse_status pse_neighbors_impl(pse_ctx *c, const float *d_pos);    // enqueue only
pse_status pse_neighbors_settle(pse_ctx *c, bool *redo);
pse_status pse_neighbors_examine(pse_ctx *c, int slot, bool *redo);
pse_status pse_neighbors_sync(pse_ctx *c, const float *d_pos);    // build + settle, repeated until complete
pse_status pse_scan_u64(pse_ctx *c, const int *d_in, unsigned long long *d_out, size_t n);   // exclusive, n+1 outputs
pse_status pse_scan_i32(pse_ctx *c, const int *d_in, int *d_out, size_t n);
pse_status pse_rank_sort(pse_ctx *c, const int *seg_start, int nseg, const int *in, int *out);
pse_status pse_get_neighbors_impl(pse_ctx *c, int *d_count, int *d_index, size_t cap, size_t *total);
pse_status pse_hs_forces_packed(pse_ctx *c, double dt, float *d_out_packed);
pse_status pse_bond_forces_orig(pse_ctx *c, float *d_F);   // [N][3], original numbering, overwritten
// realspace.cu
pse_status pse_real_init(pse_ctx *c);     // per-device kernel attributes (dynamic shared memory opt-in)
pse_status pse_real_apply(pse_ctx *c, const float *d_in, float *d_out, int mode = PSE_MODE_ALL);   // out = M_r in
// wavespace.cu
pse_status pse_wave_init(pse_ctx *c);
void pse_wave_free(pse_ctx *c);
void pse_wave_set_stream(pse_ctx *c, cudaStream_t st);    // stream of the cuFFT plans
pse_status pse_tile_bins(pse_ctx *c);
pse_status pse_particle_windows(pse_ctx *c);   // d_pbase, d_pw from d_pos (after the cell sort)
pse_status pse_wave_apply(pse_ctx *c, const float *d_in, float *d_out, bool accumulate, int mode = PSE_MODE_ALL);   // out (+)= M_w in
pse_status pse_wave_spread(pse_ctx *c, const float *d_in, int plan);                    // packed vector -> c->d_grid, planes of plan 0 / 1 / 2
pse_status pse_wave_interp(pse_ctx *c, float *d_out, bool accumulate, int oplan);      // c->d_grid -> packed vector, planes of oplan 3 / 1 / 2
pse_status pse_wave_brownian(pse_ctx *c, const float *d_noise_wave, float *d_out, bool accumulate, float *d_outW = nullptr);
// couplet.cu (torque / angular-velocity rows, NEXT-3)
void pse_couplet_free(pse_ctx *c);
void pse_build_rot_table(double a, double eta, double xi, double rcut, int ntab, std::vector<float> &tab);   // tables.cu
// krylov.cu
pse_status pse_krylov_init(pse_ctx *c);   // cooperative-grid cap of the step kernels on the context's device
pse_status pse_pack(pse_ctx *c, const float *d_F, const float *d_S, float *d_packed);      // original -> sorted
pse_status pse_pack8(pse_ctx *c, const float *d_v8, float *d_packed);
pse_status pse_unpack(pse_ctx *c, const float *d_packed, float scale, float *d_U, float *d_E);
pse_status pse_lanczos_sqrt(pse_ctx *c, const float *d_w, float *d_y, int *iters, int fixed_m = 0);          // y = M_r^{1/2} w
// the same iteration on vectors of `width` packed arrays ([width][N][8], width = 2: force/stresslet slots then torque slots) with
// any operator out = A in and work vector d_u of that size; checks convergence every iteration, leaves the iteration history alone
typedef pse_status (*pse_matvec_fn)(pse_ctx *c, const float *d_in, float *d_out);
pse_status pse_lanczos_sqrt_wide(pse_ctx *c, const float *d_w, float *d_y, int *iters, int width, pse_matvec_fn op, float *d_u);
bool pse_lanczos_validate(pse_ctx *c, int m, bool *shrink);
bool pse_gmres_validate(pse_ctx *c, int m, bool *shrink);
pse_status pse_gmres_constraint(pse_ctx *c, const float *d_Fp, const float *d_UBp, const float *d_EBp,
                                float *d_outp, int *iters, int fixed_m = 0);
pse_status pse_axpby(pse_ctx *c, size_t n, float alpha, const float *x, float beta, float *y);

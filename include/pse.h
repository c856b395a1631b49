/* pse.h — C ABI of libpse: positively-split Ewald (PSE) grand mobility with stresslets on one B200 (sm_100a).
 *
 * Method: Fiore & Swan, arXiv 1709.06946 ("PAPER.md").  Every call below cites the passage that defines it.
 *
 * Conventions
 *   - Pointers prefixed d_ are DEVICE pointers owned by the caller (e.g. torch tensors); h_ are HOST pointers.
 *     The library never frees or reallocates caller buffers.  All internal buffers belong to the context.
 *   - All work is enqueued on the CUDA stream given at pse_create (NULL = legacy default stream), on the device that was
 *     current at pse_create.  Calls that return iteration counts or need host-side convergence decisions synchronise that
 *     stream.  Callers that produce inputs on another stream must order that stream before the call themselves.
 *   - fp32 on the device.  Per-particle vectors: positions [N][4] (x,y,z,unused); forces/velocities [N][3];
 *     stresslets / rates of strain [N][5] as coordinates in the orthonormal basis of symmetric traceless tensors
 *       e1=(xx-yy)/sqrt2, e2=(2zz-xx-yy)/sqrt6, e3=(xy+yx)/sqrt2, e4=(xz+zx)/sqrt2, e5=(yz+zy)/sqrt2
 *     (the paper says only "5 for the stresslet"; reading R9).
 *   - Errors are return codes; pse_last_error gives a message.  No exceptions cross this boundary, no exit().
 *   - There is no CPU fallback: without a CUDA device every compute call returns PSE_ECUDA.
 */
#ifndef PSE_H
#define PSE_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct pse_ctx pse_ctx;

typedef enum {
    PSE_OK = 0, PSE_EINVAL = 1, PSE_ENOMEM = 2, PSE_ECUDA = 3, PSE_ECUFFT = 4, PSE_ENOTREADY = 5,
    PSE_ENOCONV = 6, PSE_EOVERFLOW = 7
} pse_status;

/* which half of the Ewald sum pse_mobility_apply evaluates (Eq. 30) */
enum { PSE_REAL = 1, PSE_WAVE = 2, PSE_BOTH = 3 };

/* Window of the spreading / interpolation operators Q, Q^T of Eq. (42) on its P^3-point support:
 *   PSE_WINDOW_GAUSS  the paper's truncated Gaussian, exp(-2 xi^2 r^2/eta_g) with eta_g = (h P xi/m)^2, m = sqrt(pi P)
 *                     (PAPER.md:263, 306, 334); needs eta_g < 1;
 *   PSE_WINDOW_ES     "exponential of semicircle" exp(beta (sqrt(1 - (2t/P)^2) - 1)), beta = 2.2 P, t = offset in grid
 *                     spacings: same support, reaches a given tolerance with fewer points (R3, R6).  Default.
 * The window is divided out exactly in wave space (R4), so the operator is the same; only the quadrature
 * error for a given P differs.  P from pse_suggest_params* fits the window it was asked for. */
enum { PSE_WINDOW_GAUSS = 0, PSE_WINDOW_ES = 1 };

/* phases reported by pse_get_timings */
enum { PSE_T_NEIGHBORS = 0, PSE_T_REAL = 1, PSE_T_SPREAD = 2, PSE_T_FFT_FWD = 3, PSE_T_SCALE = 4, PSE_T_FFT_INV = 5,
       PSE_T_INTERP = 6, PSE_T_VECTOR = 7, PSE_T_PACK = 8, PSE_T_COUNT = 9 };

/* Parameter derivation from a tolerance (reading R6; paper: eps_r ~ exp(-xi^2 rcut^2) PAPER.md:207,
 * quadrature bound Eq. (55) with m = sqrt(pi P) PAPER.md:308, 334).  Host only, no GPU needed.
 *   in : N, L, a, tol, xi
 *   out: *grid (FFT points per dimension, 2^a 3^b 5^c 7^d), *P (window support, points per dimension: 3/4/5 at
 *        tol = 1e-2/1e-3/1e-4 for PSE_WINDOW_ES, 5/6/8 for PSE_WINDOW_GAUSS), *rcut (real-space cutoff).
 *   Returns PSE_EINVAL if no valid choice exists (rcut > L/2).  pse_suggest_params = the default window. */
pse_status pse_suggest_params(int N, double L, double a, double tol, double xi, int *grid, int *P, double *rcut);
pse_status pse_suggest_params_window(int N, double L, double a, double tol, double xi, int window, int *grid, int *P, double *rcut);
/* The same for a deformed lattice A = [[a11, a12, 0], [0, a22, 0], [0, 0, 1]] (see pse_set_lattice): the grid grows by the largest
 * column norm of A (the index range that still holds every |k| <= k_cut), P does not change (the window acts on lattice
 * coordinates), and PSE_EINVAL also if rcut * (largest row norm of A^-1) > L/2 or det A != 1. */
pse_status pse_suggest_params_lattice(int N, double L, double a, double tol, double xi, int window, double a11, double a12, double a22,
                                      int *grid, int *P, double *rcut);

/* Create a context for N equal spheres of radius a in a cubic periodic box of edge L, viscosity eta, thermal
 * energy kT, splitting parameter xi (Eq. 28), FFT grid `grid`^3, window support P^3 grid points
 * (PAPER.md:227), real-space cutoff rcut, Krylov tolerance tol.  Builds the
 * real-space tables (Eqs. 25-27 PAPER.md:127-143 via DESIGN.md §3), cuFFT plans and workspaces on the current device.
 * pse_create uses PSE_WINDOW_ES; pse_create_window takes the window explicitly (no environment variable is read anywhere).
 * PSE_EINVAL: non-positive sizes, rcut > L/2, rcut < 2a, P > grid, P > 16, unknown window, and for PSE_WINDOW_GAUSS a
 * shape parameter eta_g >= 1.  *out is set even on failure so that pse_last_error works; destroy it. */
pse_status pse_create(pse_ctx **out, int N, double L, double a, double eta, double kT, double xi,
                      int grid, int P, double rcut, double tol, void *cuda_stream);
pse_status pse_create_window(pse_ctx **out, int N, double L, double a, double eta, double kT, double xi,
                             int grid, int P, double rcut, double tol, int window, void *cuda_stream);
pse_status pse_destroy(pse_ctx *ctx);

/* Deformed periodic lattice: the periodic cell is the cube of edge L mapped by the volume-preserving
 * A = [[a11, a12, 0], [0, a22, 0], [0, 0, 1]], i.e. the lattice vectors are the columns of L A.  Simple shear (Lees-Edwards,
 * Eq. 56): a11 = a22 = 1, a12 = gamma; planar extension (Kraynik-Reinelt, Eq. 58): a11 = epsilon,
 * a22 = 1/epsilon, a12 = 0; any other volume-preserving lattice in the x-y plane B (a Kraynik-Reinelt cell in the lab frame) is
 * B = Q A with A of this form and Q a rotation about z: pass A and work in the frame x' = Q^T x.  The grid grows with the longest
 * lattice vector (column of A), so describe the lattice by its shortest (Gauss-reduced) basis.  Positions, forces, velocities stay PHYSICAL (Cartesian) vectors; any periodic image of a position is
 * accepted.  Inside, particles are carried in lattice coordinates s = A^-1 x, so cells, spreading and interpolation are those of
 * the cube, separations are r = A d and wave vectors k = (2 pi/L) A^-T n (reading R22): P is that of the cube, the grid
 * must be pse_suggest_params_lattice's.  Call before pse_neighbors; the neighbour structures are invalidated; pse_step then leaves
 * positions unwrapped.  (1, 0, 1) restores the cube.  Synchronises the stream.  Cheap enough to call before every step of a flowing
 * suspension (grid taken for the largest strain): the kernels read A from device memory, so the captured graphs of pse_step survive
 * the call and are rebuilt only when the cell count of the neighbour search changes or the lattice becomes / stops being the cube.
 * PSE_EINVAL: a11 <= 0, a22 <= 0, a11 a22 != 1, or rcut * (largest row norm of A^-1) > L/2. */
pse_status pse_set_lattice(pse_ctx *ctx, double a11, double a12, double a22);

/* Bin the particles (positions may be unwrapped; they are wrapped into [0,L)) into linked cells of edge >= rcut
 * and build the full neighbour list {beta != alpha : |x_alpha - x_beta|_min-image^2 < rcut^2}, plus
 * the FFT-grid tile bins used by spread/interpolate.  Must be re-called whenever positions change.
 * d_pos: [N][4] float, device.  Synchronises once (the list size comes back to the host; inside pse_step the builds are
 * only enqueued and that read-back is examined after the Krylov solve that follows). */
pse_status pse_neighbors(pse_ctx *ctx, const float *d_pos);

/* [U;E] = M [F;S]  (Eqs. 30-31): real-space pair sum over the neighbour list with tabulated
 * functions (Eqs. 25-27) plus the spectral-Ewald wave-space sum sigma Q^T F^H P^H B P F Q (Eq. 42).
 * d_F [N][3], d_S [N][5] in; d_U [N][3], d_E [N][5] out (overwritten).  which = PSE_REAL | PSE_WAVE | PSE_BOTH.
 * PSE_ENOTREADY before pse_neighbors.  Asynchronous. */
pse_status pse_mobility_apply(pse_ctx *ctx, const float *d_F, const float *d_S, float *d_U, float *d_E, int which);

/* Brownian slip velocities [U^B;E^B] = sqrt(2 kT/dt) ( M_r^{1/2} w1 + M_w^{1/2} w2 )  (Eqs. 71, 75, 76, B4;
 * PAPER.md:409, 449, 462, 759).  M_r^{1/2} w1 by Lanczos to relative change <= tol;
 * M_w^{1/2} w2 = sigma^{1/2} Q^T F^H P^H B^{1/2} w2 with conjugate-symmetric complex noise.
 * d_noise_real: [N][8] i.i.d. N(0,1), per particle (Ux,Uy,Uz,e1..e5).
 * d_noise_wave: [3][grid][grid][grid/2+1][2] i.i.d. N(0,1); layout and conjugacy rule: DESIGN.md reading R8.
 * lanczos_iters (host, may be NULL) receives the iteration count.  Synchronises the stream. */
pse_status pse_brownian(pse_ctx *ctx, double dt, const float *d_noise_real, const float *d_noise_wave,
                        float *d_UB, float *d_EB, int *lanczos_iters);

/* Stresslet-constrained velocities at the current positions (Eqs. 36-38, 78):
 * solve M_ES S = -(E^B + M_EF F) by GMRES (relative residual <= tol), U = U^B + M_UF F + M_US S.
 * d_F [N][3] (may be NULL = 0), d_UB [N][3], d_EB [N][5] (may be NULL = 0) in; d_U [N][3], d_S [N][5] out.
 * gmres_iters (host, may be NULL).  PSE_ENOCONV if not converged in 50 iterations (best iterate written). */
pse_status pse_constrained_solve(pse_ctx *ctx, const float *d_F, const float *d_UB, const float *d_EB,
                                 float *d_U, float *d_S, int *gmres_iters);

/* The full couplet of Eq. (31): [U; Omega; E] = M [F; L; S] with the torque L and the angular velocity Omega
 * of Eqs. (32), (34) beside force, stresslet, velocity and rate of strain.  Conventions (reading R21:
 * the paper's index order in Eqs. (4)/(8)/(16) and the sign of Eq. (32) disagree with each other, so the
 * physics decides): a torque acts on the fluid as the force density (1/2) curl(L delta), Omega is the sphere average of
 * (1/2) curl u, both with the couplet shape factor 3 j1(ka)/ka: an isolated sphere turns with L/(8 pi eta a^3),
 * a torque on beta moves alpha with L x r/(8 pi eta r^3), r = x_alpha - x_beta > 2a.  The matrix stays symmetric positive
 * semi-definite; its force / stresslet block is pse_mobility_apply's.
 * d_F [N][3], d_L [N][3], d_S [N][5] in (any may be NULL = 0, not all); d_U [N][3], d_W [N][3] (Omega), d_E [N][5] out (any may
 * be NULL, not all).  which = PSE_REAL | PSE_WAVE | PSE_BOTH.  The first call allocates the torque planes (3 spectra, 3 packed
 * vectors, one table) and synchronises once; later calls are asynchronous.  PSE_ENOTREADY before pse_neighbors. */
pse_status pse_mobility_apply_full(pse_ctx *ctx, const float *d_F, const float *d_L, const float *d_S,
                                   float *d_U, float *d_W, float *d_E, int which);

/* The Brownian slip of the full couplet, script-U^B = [U^B; Omega^B] and E^B (Eq. 76 with the 11 components of Eq. 31; the paper's
 * "11" grids): sqrt(2 kT/dt) ( M_r^{1/2} w1 + M_w^{1/2} w2 ) with the 11N x 11N matrices.  The wave half draws the
 * SAME random fluid velocity field as pse_brownian from the same d_noise_wave and reads three more moments of it
 * (Omega_h = (i/2) s1 k x uh); the real half is a Lanczos iteration on the 11-component pair sum.
 * d_noise_real: [N][11] i.i.d. N(0,1), per particle (Ux,Uy,Uz, Ox,Oy,Oz, e1..e5); d_noise_wave as in pse_brownian.
 * d_UB [N][3], d_WB [N][3], d_EB [N][5] out (any may be NULL).  Synchronises the stream (every Lanczos iteration). */
pse_status pse_brownian_full(pse_ctx *ctx, double dt, const float *d_noise_real, const float *d_noise_wave,
                             float *d_UB, float *d_WB, float *d_EB, int *lanczos_iters);

/* pse_constrained_solve with torques (Eqs. 36-38, with script-F = [F; L], script-U = [U; Omega]):
 * M_ES S = -(E^B + M_EF F + M_EL L) by GMRES, then U = U^B + M_UF F + M_UL L + M_US S and Omega = M_OF F + M_OL L + M_OS S.
 * d_F, d_L, d_UB, d_EB may be NULL (= 0); d_U [N][3], d_S [N][5] out; d_W [N][3] out, may be NULL (one product less).
 * Omega^B of pse_brownian_full, if wanted, is added by the caller (it does not enter the constraint). */
pse_status pse_constrained_solve_full(pse_ctx *ctx, const float *d_F, const float *d_L, const float *d_UB, const float *d_EB,
                                      float *d_U, float *d_W, float *d_S, int *gmres_iters);

/* pse_step with external torques: one mid-point step of Eqs. (76)-(79) in which script-F = [F^P; L] carries the torques d_L [N][3]
 * (may be NULL) beside the overlap / bond forces, and script-U = [U; Omega] is returned: positions advance with U_{k+1/2}, the
 * angular velocities Omega_{k+1/2} = M_OF F + M_OL L + M_OS S go to d_W [N][3] (may be NULL) for the caller's own orientation
 * update.  The Brownian slip is pse_brownian's (no Brownian angular velocity is added; pse_brownian_full has it).  Runs the checked
 * path (synchronous builds, per-iteration convergence checks), not the graph replay of pse_step. */
pse_status pse_step_full(pse_ctx *ctx, float *d_pos, double dt, const float *d_L, const float *d_noise_real, const float *d_noise_wave,
                         float *d_W, int *gmres_iters, int *lanczos_iters);

/* Heyes-Melrose hard-sphere overlap force at the current positions (named by BASELINE.json, not the paper;
 * DESIGN.md reading R12): F_i = sum_{j: r_ij<2a} 3 pi eta a (2a - r_ij)/dt rhat_ij.  d_F [N][3] out. */
pse_status pse_hard_sphere_forces(pse_ctx *ctx, double dt, float *d_F);

/* The same force for callers that cannot call cudaMalloc (under CUDA-graph capture, in a serving loop, in a harness that
 * forbids it): no context, no allocation of any kind.  The linked-cell scratch (cell heads + per-particle links) is a
 * static __device__ array of PSE_NOALLOC_SCRATCH_BYTES (5 MiB) that every GPU holding the library keeps until exit.
 *   N <= PSE_NOALLOC_MAX_N particles (PSE_EOVERFLOW beyond, nothing is launched); L >= 4a (PSE_EINVAL: minimum image);
 *   d_pos [N][4] device, may be unwrapped; d_F [N][3] device, overwritten, original numbering; cuda_stream = the stream
 *   the three operations (clear heads, link, forces) are enqueued on, on the CURRENT device (NULL = legacy default).
 *   h_err: HOST buffer of h_err_cap bytes receiving a message on failure (may be NULL).  Asynchronous.
 * All calls share the one array: calls on one stream are ordered; calls that overlap on the GPU (two streams, two
 * threads) race and give garbage.  Nothing is kept between calls.  The first call on a device looks up the array's
 * device address (cudaGetSymbolAddress): make it before a capture begins.  The sum over overlapping partners runs
 * in a fixed order (neighbour cells, ascending particle index), so repeated calls agree bit for bit; against
 * pse_hard_sphere_forces the per-pair terms are identical and only the fp32 summation order differs. */
#define PSE_NOALLOC_MAX_N 1048576
#define PSE_NOALLOC_SCRATCH_BYTES 5242880
pse_status pse_hard_sphere_forces_noalloc(int N, double L, double a, double eta, double dt, const float *d_pos, float *d_F,
                                          void *cuda_stream, char *h_err, size_t h_err_cap);

/* Bonds with the pair potential U(r) = k |r - r0| of the paper's equilibrium test (its Boltzmann
 * distribution of r is Eq. (80)).  h_pairs: HOST array [n_bonds][2] of particle indices (copied);
 * n_bonds = 0 removes all bonds.  pse_step adds the bond forces, evaluated at x_{k+1/2} with the minimum image, to F^P.
 * Synchronises the stream.  PSE_EINVAL: index out of range, i == j, r0 < 0. */
pse_status pse_set_bonds(pse_ctx *ctx, const int *h_pairs, int n_bonds, double k, double r0);
/* Bond forces at the positions of the last pse_neighbors call: F_i = -k sign(r - r0) rhat_ij, F_j = -F_i,
 * rhat_ij = (x_i - x_j)/r.  d_F [N][3] out (overwritten; zero without bonds).  Asynchronous. */
pse_status pse_bond_forces(pse_ctx *ctx, float *d_F);

/* One mid-point step of the constrained overdamped Langevin dynamics, Eqs. (76)-(79):
 * neighbours(x_k); Brownian slip; x_{k+1/2} = x_k + dt/2 U^B; neighbours(x_{k+1/2}); hard-sphere (+ bond) forces;
 * constrained solve; x_{k+1} = x_k + dt U_{k+1/2} (wrapped into [0,L)).  d_pos [N][4] in/out.
 * On return the context's neighbour structures refer to x_{k+1/2}; call pse_neighbors before further products. */
pse_status pse_step(pse_ctx *ctx, float *d_pos, double dt, const float *d_noise_real, const float *d_noise_wave,
                    int *gmres_iters, int *lanczos_iters);

/* End-to-end variants with HOST buffers (pinned or pageable): the library copies inputs host->device, runs the
 * device call of the same name, copies the results device->host and synchronises.  These are what bench.py's
 * "e2e" number times.  h_pos [N][4] (in/out for pse_step_host), h_F [N][3], h_S [N][5], h_U [N][3], h_E [N][5],
 * h_noise_real [N][8], h_noise_wave [3][grid][grid][grid/2+1][2]. */
pse_status pse_mobility_apply_host(pse_ctx *ctx, const float *h_pos, const float *h_F, const float *h_S,
                                   float *h_U, float *h_E);
pse_status pse_step_host(pse_ctx *ctx, float *h_pos, double dt, const float *h_noise_real, const float *h_noise_wave,
                         int *gmres_iters, int *lanczos_iters);

/* Introspection for the parity tests and the harness. */
/* Neighbour list in ORIGINAL particle numbering: d_count [N]; d_index holds the lists of particle 0,1,...
 * concatenated (offsets = exclusive scan of d_count); order within a list is unspecified.  *total (host) gets
 * the number of entries; if cap < total only *total is written (PSE_EOVERFLOW).  d_index may be NULL. */
pse_status pse_get_neighbors(pse_ctx *ctx, int *d_count, int *d_index, size_t cap, size_t *total);
/* Switch per-phase CUDA-event timing on/off (adds event records, no synchronisation until read). */
pse_status pse_set_profiling(pse_ctx *ctx, int on);
/* Accumulated per-phase milliseconds and launch counts since the last call (synchronises); arrays of n entries. */
pse_status pse_get_timings(pse_ctx *ctx, float *h_ms, int *h_launches, int n);
/* Number of kernels (own + cuFFT calls) enqueued since pse_create. */
long long pse_kernel_launches(const pse_ctx *ctx);
/* Copy the fp32 real-space table to the host: n nodes x 8 (F1,F2,G1+G2,G1+4G2,A,B,D,0), node i at r = i*dr. */
pse_status pse_get_table(pse_ctx *ctx, float *h_table, int cap_nodes, int *n_nodes, double *dr);
const char *pse_last_error(const pse_ctx *ctx);
const char *pse_version(void);

#ifdef __cplusplus
}
#endif
#endif

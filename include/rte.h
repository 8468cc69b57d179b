/* rte.h — C ABI of the B200-native pseudospectral P_N radiative-transport time stepper.
 *
 * The library advances the spherical-harmonic (3-D) / circular-harmonic (2-D) moment fields psi_c(r,t) of the
 * radiative transport equation (eq.(1)) on a periodic Fourier-collocation grid:
 *
 *     psi_c^{n+1}(r) = psi_c^n(r) - c dt ( T_c(r) + sigma_l(r) psi_c^n(r) ) + c dt 1_Omega(r) q_c(r, t_n)
 *
 *     T      = sum_axis A_axis D_axis psi        streaming operator s.grad of eq.(6)/(10)
 *     D_axis = IDFT_axis( i k_axis DFT_axis(.) ) spectral derivative, eq.(7)-(8)
 *     sigma_l= mu_a + mu_s (1 - g^l)  in Omega   Henyey-Greenstein diagonal mu_t - mu_s g^l, eq.(5),(9)
 *            = mu_b                   in the PML eq.(12); half-cosine profile of PAPER.md:165
 *     step   = forward Euler                     eq.(11), PAPER.md:104 (signs per DESIGN.md reading R3)
 *
 * All of it runs in hand-written sm_100a kernels; there is no CPU fallback: every call that needs the device
 * returns RTE_ECUDA when no CUDA device / wrong architecture is present.
 *
 * Conventions
 *   units            mm, ps, mm^-1 (as the paper)
 *   grid             nx*ny*nz cells, x fastest; cell i along an axis sits at (i - n/2) dx; nz = 1 when dim = 2.
 *                    Every extent must be an EVEN number of the form 2^a 3^b in [16, 1024] (16, 18, 24, 32, 36, 48, 54,
 *                    64, 72, 96, 108, 128, 144, 162, 192, 216, 256, 288, 324, 384, 432, 486, 512, 576, 648, 768, 864,
 *                    972, 1024), and one pencil of all coefficients must fit a shared-memory tile
 *                    (n * 8 * ceil(C/2) bytes + the diagonal table <= 226 KB; else RTE_EUNSUPPORTED).
 *   order            1 <= N <= 31 (at most 1024 coefficients in 3-D); larger N is RTE_EINVAL / a negative count.
 *   coefficients     3-D: C=(N+1)^2, c = l*l + l + m; m>=0 is the cos-type real harmonic a_l^m, m<0 the sin-type
 *                    b_l^|m| (R6).  2-D: C=2N+1, c=0 -> a_0, c=2m-1 -> a_m, c=2m -> b_m (R8).
 *                    Coefficient 0 is the fluence in both (R9).
 *   field layout     external arrays are [c][z][y][x] fp32, contiguous (x fastest).
 *   pointers         "_dev" arguments are CUDA device pointers (e.g. torch.Tensor.data_ptr()) valid on the context's
 *                    device; "_host" arguments are host pointers (pinned memory makes the copies asynchronous).
 *                    Every call on a context must be made with the CUDA device that was current at rte_create.
 *                    The library never frees caller memory.  It keeps the workspace and the stream until
 *                    rte_destroy; every other array is consumed (stream-ordered) during the call.
 *   stream           all work is enqueued on the cudaStream_t passed to rte_create (NULL = legacy default
 *                    stream); calls return without synchronising unless stated.
 *   errors           every function returns an rte status; nothing throws or aborts across the ABI.
 *                    rte_last_error gives a text for the last failure on that context.
 */
#ifndef RTE_H_
#define RTE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rte_ctx rte_ctx; /* opaque; owned by the library, freed by rte_destroy */

enum { RTE_OK = 0, RTE_EINVAL = 1, RTE_ENOMEM = 2, RTE_ECUDA = 3, RTE_ESTATE = 4, RTE_EUNSUPPORTED = 5 };

typedef struct {
    int dim;        /* 2 or 3 */
    int nx, ny, nz; /* nz = 1 when dim = 2 */
} rte_grid;

/* Perfectly matched layer, eq.(12) PAPER.md:113-119.  width = cells per side (0 = fully periodic, no layer).
 * Depth of cell i along an axis: p = max(width - i, i - (n-1-width), 0); delta = max over axes of p / width;
 * mu_b = mu_lo + (mu_hi - mu_lo) (1 - cos(pi delta))/2 for delta > 0 (half-cosine; R11).
 * In the layer sigma_l = mu_b for every l, mu_s = 0 and q = 0.  Requires 2*width < every extent. */
typedef struct {
    int width;
    float mu_lo, mu_hi; /* mm^-1 */
} rte_pml;

/* Optical properties of eq.(1)-(2).  Each pointer is a DEVICE pointer to either 1 value (is_map = 0) or
 * nx*ny*nz values in [z][y][x] order (is_map = 1).  Values inside the PML are ignored. */
typedef struct {
    const float *mu_a, *mu_s, *g;
    int mu_a_is_map, mu_s_is_map, g_is_map;
} rte_media;

/* ---- host-only helpers (no device needed) ------------------------------------------------------------------ */

/* Number of real coefficient fields C: (N+1)^2 in 3-D, 2N+1 in 2-D (R8). <0 on bad input. */
int rte_num_coeffs(int dim, int N);

/* Real-basis streaming coupling of eq.(6)/(10) (R1, R7, R8):
 * A_out[c*C + c'] (host, C*C doubles) with T_c = sum_c' A[c][c'] d psi_c' / d x_axis; axis 0=x, 1=y, 2=z. */
int rte_coupling_table(int dim, int N, int axis, double* A_out_host);

/* Internal storage layout (host only; no device call).  The C fields are stored cell-major in Cp = 2*P slots, two
 * real fields per "pair" (one complex FFT differentiates both).  The position of each pair
 * in a cell record and the order of its coupling entries are chosen to make the kernels' shared-memory gathers
 * bank-conflict free.  Outputs (any may be NULL): Cp_out = number of slots; ext_of_slot_host[Cp] = external
 * coefficient index stored in each slot, -1 for a zero pad slot (slot 0 is always coefficient 0, the fluence);
 * cost_host[3] = modelled gather wavefronts {natural order, chosen layout, conflict-free ideal}.
 * Returns RTE_EINVAL for dim not in {2,3} or N < 1. */
int rte_storage_layout(int dim, int N, int* Cp_out, int* ext_of_slot_host, int* cost_host);

/* Bytes of device workspace rte_create needs for this grid and order (two state buffers — the step reads one and
 * accumulates the next state into the other, then they trade places — and three per-cell coefficient maps). */
int rte_workspace_bytes(const rte_grid* grid, int N, size_t* bytes_out);

/* Bytes of n_fields additional state-sized device buffers (caller-owned, handed over with rte_set_extra_workspace):
 * rte_step_ssprk3 needs 1 field, rte_apply_operator 2, rte_solve_steady restart + 3 (+ 3 with its preconditioner). */
int rte_extra_workspace_bytes(const rte_grid* grid, int N, int n_fields, size_t* bytes_out);

/* Forward-Euler stability bound of the step eq.(11) (R10; the paper picks dt "by inspection", PAPER.md:141,
 * "time-steps of the order of 100 fs provide stability").  Forward Euler is stabilised only by the
 * scattering damping: for every Fourier mode the eigenvalues lambda of M(k) = -c (i k A + diag sigma_l),
 * sigma_l = mu_a + mu_s (1 - g^l), must satisfy dt <= -2 Re(lambda) / |lambda|^2.  The bound is evaluated on 200
 * wavenumber magnitudes up to the corner Nyquist sqrt(dim) (pi/dx)(1 - 2/n_min) (k along one axis: rotational
 * invariance) for ONE medium — pass the weakest damping present: smallest mu_a and mu_s, largest g.
 * bound_ps_out: the bound; dt_ps_out: the recommended step, half of it (a PML moves the true bound by x0.7-2).
 * Either output may be NULL.  Host only. */
int rte_stable_dt(int dim, int N, int n_min, float dx_mm, float c_mm_per_ps, float mu_a_min, float mu_s_min,
                  float g_max, double* bound_ps_out, double* dt_ps_out);

/* ---- life cycle ---------------------------------------------------------------------------------------------- */

/* Build a solver: validates, generates the coupling tables, wavenumbers (k at Nyquist = 0, R5), FFT
 * twiddles and the per-cell sigma / PML maps on the device, zeroes the state, sets t = 0.
 * workspace_dev: caller-owned device memory of at least rte_workspace_bytes, 256-byte aligned, alive until
 * rte_destroy.  cuda_stream: a cudaStream_t (may be NULL).
 * RTE_EINVAL: N<1 or N>31, dx/dt/c <= 0, unsupported extent, dim/grid mismatch, PML too wide, workspace too small or
 * misaligned.  RTE_EUNSUPPORTED: a pencil of all coefficients does not fit one shared-memory tile.  RTE_ECUDA: no sm_100 device or a CUDA failure.  The time step is NOT checked for stability
 * (the paper chooses dt "by inspection"). */
int rte_create(rte_ctx** out, const rte_grid* grid, int N, float dx_mm, float dt_ps, float c_mm_per_ps,
               const rte_media* media, const rte_pml* pml, void* workspace_dev, size_t workspace_bytes,
               void* cuda_stream);
void rte_destroy(rte_ctx* ctx);

/* ---- state ----------------------------------------------------------------------------------------------------- */

/* Set / read all moment fields, [C][nz][ny][nx] fp32.  An initial radiance distribution is how a delta(t) pulse
 * enters.  rte_set_state does not reset the clock; rte_reset_time does. */
int rte_set_state(rte_ctx* ctx, const float* psi_dev);
int rte_get_state(rte_ctx* ctx, float* psi_dev);
int rte_set_state_host(rte_ctx* ctx, const float* psi_host); /* host -> device inside the call, stream-ordered */
int rte_get_state_host(rte_ctx* ctx, float* psi_host);       /* device -> host, synchronises the stream       */
int rte_reset_time(rte_ctx* ctx);

/* Source term q_c(r,t) = w[c] * S(r) * f(t) of eq.(1),(4), added as c dt q(t_n) each step
 * (eq.(11); R3, R14) and only inside Omega (eq.(12)).
 * w_host: C angular weights (host).  S: spatial footprint on the box [origin, origin+extent) in cells, laid out
 * [bz][by][bx]; *_dev takes a device pointer, *_host a host pointer.  temporal_kind: 0 none (clears the source),
 * 1 constant f = 1, 2 Gaussian f = exp(-(t-t0)^2 / (2 sigma_t^2)). */
int rte_set_source(rte_ctx* ctx, const float* w_host, const float* S_dev, const int box_origin[3],
                   const int box_extent[3], int temporal_kind, float t0_ps, float sigma_t_ps);
int rte_set_source_host(rte_ctx* ctx, const float* w_host, const float* S_host, const int box_origin[3],
                        const int box_extent[3], int temporal_kind, float t0_ps, float sigma_t_ps);

/* ---- the hot path ---------------------------------------------------------------------------------------------- */

/* Advance nsteps forward-Euler steps (eq.(11)); asynchronous on the stream.  One step = one pencil-FFT
 * kernel per axis (coupling -> DFT -> i k -> IDFT, eq.(6)-(10)): the x kernel also applies scattering, PML and source
 * (eq.(9),(12)) and stores psi(1 - c dt sigma_l) + c dt q - c dt T_x into the second state buffer, the other axes add
 * their -c dt T_a to it; the buffers then trade places.  Results are bit-reproducible from run to run.
 * Grids whose state is at most 24 MB (L2-resident, launch-bound) replay the same launches from a CUDA graph, 32 steps
 * per replay (captured on a private stream by the first call that asks for >= 4 steps; the caller's stream must not be
 * capturing then); the results are identical to the eager path.  Grids without specialised kernels (anything but the BASELINE
 * shapes) time a few block sizes per axis at the context's first sweep and keep the fastest: that first call synchronises
 * the stream once; results do not depend on the choice. */
int rte_step(rte_ctx* ctx, int nsteps);

/* Hand the library additional caller-owned device memory (256-byte aligned; rte_extra_workspace_bytes) that it keeps
 * until rte_destroy or the next call of this function (extra_dev = NULL takes it back).  Synchronises the stream. */
int rte_set_extra_workspace(rte_ctx* ctx, void* extra_dev, size_t bytes);

/* NOT eq.(11): nsteps steps of the exponential (integrating-factor) Euler scheme, the family PAPER.md:109 and :195
 * point to ("exponential integrators").  The diagonal part of eq.(9) is integrated exactly, the
 * streaming term explicitly, the source through phi_1:
 *     psi^{n+1} = E (psi^n - c dt T[psi^n]) + Phi c dt q(t_n),   E = exp(-c dt sigma_l),  Phi = (1 - E)/(c dt sigma_l).
 * A uniform field decays as exp(-c sigma_l t) with no O(dt) error, also in the PML, and the stiff diagonal
 * (c dt sigma_l > 2, where eq.(11) diverges) no longer bounds dt; the streaming bound (rte_stable_dt) is unchanged to
 * leading order.  Grids with specialised kernels (the BASELINE configurations): the three specialised passes compute
 * -c dt T, one pointwise kernel applies E, Phi and the source; every other grid: fused into the generic kernels.
 * Asynchronous on the stream. */
int rte_step_exp(rte_ctx* ctx, int nsteps);

/* The time-independent transport operator of eq.(9): y = L x = T[x] + sigma_l x, so that eq.(9) reads
 * d psi/dt = -c L psi + c q and a steady state satisfies L psi = q ("repeated application of the implicit operator",
 * PAPER.md:109).  x_dev, y_dev: [C][nz][ny][nx] fp32 device arrays.  The state and the clock are untouched.
 * Needs 2 fields of extra workspace.  Asynchronous on the stream. */
int rte_apply_operator(rte_ctx* ctx, const float* x_dev, float* y_dev);

/* Steady state L psi = q (q = the source of rte_set_source with temporal factor 1) by restarted GMRES(restart),
 * entirely on the device (the paper's Krylov solver was bound by host<->device
 * transfers).  The current state is the initial guess and becomes the solution.  Stops when the TRUE relative
 * residual ||q - L psi|| / ||q||, recomputed at every restart, is <= tol, after max_restarts cycles, or when that
 * residual has improved by less than 10 % over three cycles (the fp32 floor, typically 1e-6 .. 1e-5) — neither is an
 * error: check *relres_out.  The Krylov basis, the Hessenberg matrix and the rotations live in device memory;
 * dot products / updates are this library's kernels; the host reads a few scalars once per restart cycle.
 *   precond_steps = 0: GMRES on L itself.
 *   precond_steps = s > 0: GMRES on the time-stepping fixed-point equation  (I - Phi^s) psi = Phi^s(0; q),  Phi = one
 *     SSP-RK3 step of size precond_dt_ps of d psi/dt = -c L psi + c q (the rte_step_ssprk3 map; stable up to ~ dx/c).
 *     Its fixed point is the same steady state; s steps damp every fast mode, so the Krylov space only has to resolve
 *     the few slow (diffusive) ones — far fewer basis vectors per operator sweep.
 * Extra workspace: restart + 3 fields (+ 3 more with a preconditioner); 1 <= restart <= 64.
 * applications_out: sweeps of the three pass kernels performed (one per application of L, three per RK3 step);
 * relres_out: final true relative residual (either may be NULL).  Synchronises the stream. */
int rte_solve_steady(rte_ctx* ctx, int restart, double tol, int max_restarts, int precond_steps, float precond_dt_ps,
                     int* applications_out, double* relres_out);

/* NOT the paper's integrator (the paper uses forward Euler and names better integrators as future work,
 * PAPER.md:109,195): nsteps steps of the three-stage, third-order strong-stability-preserving Runge-Kutta scheme
 * (Shu-Osher form) built from the same Euler update E(u; t) = u + dt F(u, t) of eq.(9):
 *   u1 = E(u^n; t_n),  u2 = 3/4 u^n + 1/4 E(u1; t_n + dt),  u^{n+1} = 1/3 u^n + 2/3 E(u2; t_n + dt/2).
 * Its stability region contains the imaginary axis up to sqrt(3), so dt may approach dx/c instead of the
 * scattering-limited Euler bound (R10).  Three Euler updates (9 pass kernels in 3-D); the two convex combinations
 * are fused into them (the tables of stages 2 and 3 carry the factors 1/4 and 2/3, their first pass adds 3/4 and 1/3 of u^n
 * while it stores).  Needs 1 field of extra workspace (rte_set_extra_workspace), RTE_EINVAL without it.
 * Asynchronous on the stream; rte_time_ps advances by dt per step. */
int rte_step_ssprk3(rte_ctx* ctx, int nsteps);

/* Same as rte_step, but brackets every per-axis kernel with CUDA events on the context's stream and returns the
 * accumulated device time per axis in milliseconds (ms_axis_host[3], host; unused axes get 0) and the number of
 * launches per axis actually timed (may be NULL).  Synchronises the stream before returning. */
int rte_step_profile(rte_ctx* ctx, int nsteps, double* ms_axis_host, long long* launches_axis_host);

/* Fluence Phi(r) = coefficient 0 (eq.(3) normalisation; R9) over the whole grid, PML
 * cells included, [nz][ny][nx] fp32. */
int rte_fluence(rte_ctx* ctx, float* phi_dev);
int rte_fluence_host(rte_ctx* ctx, float* phi_host); /* device -> host, synchronises the stream */

/* Relative L2 change of the fluence over Omega since the previous call of this function (inf on the first call):
 * the steady-state test of configs[3] (R17).  Synchronises the stream. */
int rte_fluence_change(rte_ctx* ctx, double* rel_change_out);

/* Instability / NaN guard (R10; the step itself never checks its time step, as in the paper):
 * energy_out = sum_c w_l ||psi_c||_2^2 over the whole grid with w_l = 2l+1 (3-D) or 1 (m = 0), 2 (m >= 1) (2-D) — the norm in
 * which the streaming operator is skew-adjoint, so in source-free stretches a stable run never lets it grow — and
 * nonfinite_out = the number of NaN / Inf values in the state (they are left out of the sum).  Either may be NULL.
 * Synchronises the stream. */
int rte_energy(rte_ctx* ctx, double* energy_out, long long* nonfinite_out);

int rte_time_ps(const rte_ctx* ctx, double* t_out);  /* t = steps taken since the last reset * dt */
int rte_sync(rte_ctx* ctx);                          /* stream synchronise; surfaces deferred CUDA errors */
const char* rte_last_error(const rte_ctx* ctx);      /* ctx may be NULL: text of the last failed rte_create */

/* Number of kernels the library has launched on this context so far (bench.py's gpu_launches claim). */
int rte_launch_count(const rte_ctx* ctx, long long* count_out);

/* ---- geometry / coefficient layer (device generators for heterogeneous media; north_star item (3)) ------------- */

/* Fill mu_a/mu_s/g maps ([z][y][x], device) with a background and n_ell axis-aligned ellipsoids (disks in 2-D),
 * later ones overwriting earlier ones.  ell_host: n_ell rows of 9 floats
 * {cx, cy, cz, ax, ay, az, mu_a, mu_s, g}: centre and semi-axes in mm in the grid frame (cell i at (i-n/2) dx).
 * A cell belongs to an ellipsoid when sum ((r-c)/a)^2 <= 1 (z term dropped in 2-D).  Any of the three output
 * pointers may be NULL. */
int rte_media_ellipsoids(const rte_grid* grid, float dx_mm, const float background[3], int n_ell,
                         const float* ell_host, float* mu_a_dev, float* mu_s_dev, float* g_dev, void* cuda_stream);

/* Smooth log-normal field: out = exp(ln(mean) - sigma_log^2/2 + sigma_log f), f = unit-variance periodic Gaussian
 * random field with covariance exp(-r^2/(2 corr_len^2)): white noise (counter-based generator)
 * circularly convolved with a separable Gaussian of std corr_len/sqrt2 per axis, renormalised to unit sample
 * variance.  scratch_dev: nx*ny*nz floats of device scratch. */
int rte_media_lognormal(const rte_grid* grid, float dx_mm, uint64_t seed, float mean, float sigma_log,
                        float corr_len_mm, float* out_dev, float* scratch_dev, void* cuda_stream);

/* rte_media_lognormal for callers that cannot allocate device memory (CUDA-graph capture, serving loops, harnesses that
 * forbid cudaMalloc): same field, same kernels, but the blur scratch and the reduction scalars live in one static device
 * array inside the library (8 MiB + 256 B per GPU, held from library load until exit) instead of caller scratch and a
 * cudaMalloc.  Calls no cudaMalloc / cudaFree / allocating routine and does not synchronise: asynchronous on the stream.
 * Limit: nx*ny*nz <= 2 097 152 cells (128^3); larger grids return RTE_EUNSUPPORTED (text in rte_last_error(NULL)).
 * All calls on one GPU share that array: calls that overlap on the GPU (different streams) race — serialise them.  The
 * array keeps the previous call's contents; the entry point clears what must start at zero itself.  (The first call
 * on a device resolves the array's address with cudaGetSymbolAddress: make it outside a capture.) */
int rte_media_lognormal_noalloc(const rte_grid* grid, float dx_mm, uint64_t seed, float mean, float sigma_log,
                                float corr_len_mm, float* out_dev, void* cuda_stream);

/* The PML profile alone (mu_b per cell, 0 inside Omega) and the Omega mask (1 inside), device outputs. */
int rte_pml_profile(const rte_grid* grid, const rte_pml* pml, float* mu_b_dev, unsigned char* inside_dev,
                    void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* RTE_H_ */

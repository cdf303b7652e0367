/* ns.h -- C ABI of libns: batched pseudo-spectral Navier-Stokes right-hand side and SSP-RK3 step
 * on the periodic torus [0,2pi)^3, hand-written CUDA for one NVIDIA B200 (sm_100a).
 *
 * Method: Rohner & Mishra, "Efficient Computation of Large-Scale Statistical Solutions to
 * Incompressible Fluid Flows", PASC'24 (arXiv 2401.09843); cited as PAPER.md:Lnnn.
 *   state              divergence-free velocity, spectral hyperviscosity discretisation
 *                      eq. (2.1)-(2.4)
 *   right-hand side    Algorithm 2 (pad 3/2, inverse FFT, u (x) u, forward FFT, dealias) and the
 *                      Leray-projected time derivative eq. (2.5)
 *   time step          third-order SSP Runge-Kutta eq. (2.6)
 *   batch              Monte-Carlo samples of Algorithm 1 evolve independently;
 *                      here they are the leading `batch` index of every array and launch
 *   outputs            "writers" of PAPER.md:L157-167: full field, energy spectrum
 * Readings of points the paper leaves open (Nyquist planes, form of Q_k, CFL formula, ...) are
 * listed in DESIGN.md section 3 (A1..A20).
 *
 * Conventions
 *   N         grid points per axis: any even N, 16 <= N <= 640.  The transforms run on a TRANSFORM GRID Nt >= N of the form
 *             p 2^a, p in {1, 3, 5, 7, 15}, Nt/2 a multiple of 8 (fp32: 16), with the padded grid M = 3 Nt / 2 >= 3N/2 -- the
 *             paper's "round the padded size up to the next 2^a 3^b 5^c 7^d"; Nt = N whenever N has that form
 *             (all BASELINE.json sizes), else the next such size or the one ns_autotune measured.  The state is truncated to
 *             the user's N (P_N of eq. 2.1) and all public arrays have the user's N; results do not depend on Nt beyond
 *             round-off, except max|u| (ns_max_velocity, the CFL step), which is a maximum over the M^3 points of the
 *             padded grid in use (ns_padded_size).
 *   spectral  complex interleaved (re,im) of `dtype`, shape [batch][3][N][N][N/2+1], index
 *             [b][component][ikx][iky][ikz], ikz fastest (r2c half spectrum, kz >= 0).
 *             Stored index i <-> wavenumber k = i (i < N/2) or i - N (i > N/2).  Coefficients are
 *             NORMALISED: u(x) = sum_k u_hat(k) e^{i k.x}.  Entries with any index == N/2 (Nyquist
 *             planes) are zero in the state and in every result (reading A3).
 *   physical  reals of `dtype`, shape [batch][3][N][N][N], index [b][component][ix][iy][iz],
 *             x_j = 2 pi j / N.
 *   memspace  every caller buffer is tagged NS_HOST (pageable or pinned host memory) or NS_DEVICE
 *             (device memory of the solver's GPU).  The caller owns every buffer it passes; the
 *             library never frees or retains it past the call.  The library owns the handle and
 *             all workspaces.
 *   stream    all work is enqueued on the cudaStream_t given to ns_create (cast to void*; NULL =
 *             the legacy default stream).  Calls that return data to NS_HOST memory, or return
 *             host scalars, synchronise that stream before returning; all others are asynchronous.
 *   errors    every int-returning call returns NS_OK (0) or a negative ns_status; the message is
 *             available from ns_last_error(h) until the next call on h.  On error the state is
 *             unchanged unless stated.  There is no CPU fallback: without a usable CUDA device
 *             ns_create fails with NS_ERR_CUDA.
 *   non-finite states   every step evaluates max|u| over the padded grid on the device (a by-product
 *             of the first stage).  A sample whose field contains NaN or inf is marked, frozen
 *             (dt_b = 0: it is never advanced again) and reported as NS_ERR_NONFINITE with its index
 *             by the next call that synchronises anyway: ns_step_cfl with dt_out, ns_step_dts,
 *             ns_advance (which stops instead of running to max_steps) and ns_max_velocity (which
 *             still fills umax_out, +inf or NaN for that sample).  Setting a new state clears the mark.
 *   threads   handles are independent; one handle must not be used concurrently.  The only process-wide state is read-mostly and
 *             mutex-protected: the ns_autotune table (device, N, dtype) -> transform grid, and the per-(kernel, device) record
 *             of function attributes already set.
 */
#ifndef NS_H_
#define NS_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ns_solver ns_solver; /* opaque */

typedef enum { NS_F64 = 0, NS_F32 = 1 } ns_dtype;
typedef enum { NS_HOST = 0, NS_DEVICE = 1 } ns_memspace;

typedef enum {
  NS_OK = 0,
  NS_ERR_INVALID_ARG = -1, /* bad N / batch / dtype / NULL pointer / nbins < 1 / bad params */
  NS_ERR_OOM = -2,         /* device allocation failed */
  NS_ERR_CUDA = -3,        /* CUDA runtime error; text in ns_last_error */
  NS_ERR_STATE = -4,       /* ns_rhs / ns_step / getters called before an initial state was set */
  NS_ERR_NONFINITE = -5    /* a sample's velocity field contains NaN or inf; ns_last_error names the sample */
} ns_status;

/* Dissipation operator of eq. (2.1)-(2.4), applied explicitly inside the RHS:
 *   d_k = nu |k|^2 + eps_N |k|^(2s) Q_k,   eps_N = eps / N^(2s-1),
 *   Q_k = 0 for |k| <= m_N, else (q_sharp ? 1 : 1 - (m_N/|k|)^q_exp),   |k| Euclidean. */
typedef struct {
  double nu;    /* Laplacian viscosity (0 disables)                                         */
  double eps;   /* hyperviscosity constant, eps_N = eps / N^(2s-1) (0 disables)              */
  double s;     /* hyperviscosity order s >= 1, may be fractional (paper uses 1 and 1.5)     */
  double m_cut; /* cutoff m_N in wavenumber units; < 0 selects sqrt(N)  (theta = 1/2)        */
  double q_exp; /* exponent (2s-1)/theta of eq. (2.3); < 0 selects (2s-1)/0.5                */
  int q_sharp;  /* 0: smooth lower bound of eq. (2.3);  1: Q_k = 1 above the cutoff          */
} ns_params;

/* Create a solver for `batch` independent samples on an N^3 grid.  `p` may be NULL (inviscid).
 * Allocates one device arena of about 15.7 * batch * Nt^3 * sizeof(complex) bytes (Nt = the transform grid; state, stage
 * state and three workspaces aliased across the passes, cf. "Workspaces", PAPER.md:L207-213;
 * ns_device_bytes returns the exact figure).
 * cuda_stream: a cudaStream_t cast to void* (NULL = default stream). */
int ns_create(ns_solver** out, int N, int batch, const ns_params* p, ns_dtype dtype, void* cuda_stream);

/* Transform-grid benchmark of PAPER.md:L175 ("On any new system, we therefore once run a benchmark of only the Fourier transform
 * storing its results and extracting the optimal padding size ... If no suitable size is found in the benchmark results, we choose
 * the next larger N with prime factors at most 7 instead"): times the transform passes a1..a6 of one sample on the first `ncand`
 * (1..16) admissible transform grids Nt >= N of the current device and records the fastest in a process-wide table keyed by
 * (device, N, dtype), which later ns_create calls for that N use; without an entry ns_create takes the first admissible Nt.
 * grids_out[ncand], ms_out[ncand] (host, may be NULL): the candidates and their milliseconds per pass sequence (0 past the
 * last candidate that exists or fits in memory); *best_out (may be NULL): the grid recorded.  Synchronous; thread safe. */
int ns_autotune(int N, ns_dtype dtype, int ncand, int* grids_out, double* ms_out, int* best_out);
/* The transform grid Nt and the padded grid M = 3 Nt / 2 of a handle (0 for NULL). */
int ns_transform_grid(const ns_solver* h);
int ns_padded_size(const ns_solver* h);
int ns_destroy(ns_solver* h);

/* Set the state from PHYSICAL samples u_phys [batch][3][N][N][N] (eq. 2.1 third line,
 * PAPER.md:L98, u(0) = P_N u_0): analysis transform with 1/N^3, Nyquist planes zeroed, Leray
 * projector (eq. 2.5) applied for k != 0, mean mode kept.  Resets every sample's time to 0. */
int ns_set_initial(ns_solver* h, const void* u_phys, ns_memspace ms);
/* Set / get the state in SPECTRAL form, no projection (Nyquist planes are zeroed on set).
 * Round trip get -> set is bit exact.  ns_set_spectral does not change the sample times. */
int ns_set_spectral(ns_solver* h, const void* u_hat, ns_memspace ms);
int ns_get_spectral(ns_solver* h, void* u_hat_out, ns_memspace ms);

/* rhs_hat_out = R(state) = (1 - k k^T/|k|^2)(-i k^T F[u (x) u]_k) - d_k u_hat_k  (Algorithm 2 +
 * eq. 2.5 + viscous term of eq. 2.1), spectral layout; R(0) = 0.  The state is unchanged. */
int ns_rhs(ns_solver* h, void* rhs_hat_out, ns_memspace ms);

/* One SSP-RK3 step (eq. 2.6) with the same dt for all samples; t_b += dt. */
int ns_step(ns_solver* h, double dt);
/* One SSP-RK3 step with a per-sample CFL step (reading A10; PAPER.md:L155 names the condition):
 *   dt_b = min(cfl * (2 pi / N) / umax_b, t_end - t_b),  umax_b = max over the padded grid of |u|_2
 * at the start of the step, evaluated on the device (no host round trip inside the step).
 * Samples with t_b >= t_end are left untouched (bit exact).  dt_out: host array [batch] or NULL;
 * when non-NULL the stream is synchronised and the steps actually taken are returned. */
int ns_step_cfl(ns_solver* h, double cfl, double t_end, double* dt_out);
/* One SSP-RK3 step with caller-given per-sample steps dt[batch] (host array); dt_b == 0 leaves
 * sample b untouched.  Used to replay a recorded CFL sequence. */
int ns_step_dts(ns_solver* h, const double* dt);
/* Integrate every sample to t_end (Algorithm 1 line "evolve the sample"; BASELINE configs[3]:
 * "integrated to t=1 at CFL 0.2"): repeated ns_step_cfl(cfl, t_end) without a host round trip per step; the host
 * reads the sample times every fourth step and stops when all have reached t_end or after max_steps steps.
 * *steps_done (may be NULL) = RK3 steps launched; steps issued after a sample has finished leave it untouched.
 * NS_ERR_INVALID_ARG for cfl <= 0 or max_steps < 0. */
int ns_advance(ns_solver* h, double cfl, double t_end, int max_steps, int* steps_done);

/* umax_out[batch] (host): max over the padded M^3 grid (M = ns_padded_size(h)) of the Euclidean |u| of the current state. */
int ns_max_velocity(ns_solver* h, double* umax_out);
/* Physical velocity on the N grid, [batch][3][N][N][N] (the "whole flow field" writer). */
int ns_get_fields(ns_solver* h, void* u_phys_out, ns_memspace ms);
/* Shell energy spectrum (reading A14):
 *   E_out[b][K] = 1/2 sum_{K-1/2 <= |k| < K+1/2} |u_hat_k|^2 over the full spectrum, K = 0..nbins-1,
 * host array [batch][nbins] of double; sum_K E = 1/2 <|u|^2> when nbins covers all modes. */
int ns_energy_spectrum(ns_solver* h, double* E_out, int nbins);
/* Shell enstrophy spectrum (the "enstrophy spectrum" writer; reading A20): with omega_hat = i k x u_hat,
 *   Z_out[b][K] = 1/2 sum_{K-1/2 <= |k| < K+1/2} |omega_hat_k|^2, same shells, weights, layout and errors as
 * ns_energy_spectrum; sum_K Z = 1/2 <|curl u|^2>. */
int ns_enstrophy_spectrum(ns_solver* h, double* Z_out, int nbins);
/* Second-order longitudinal+transverse structure function on the N grid (reading A15):
 *   S_out[b][l-1] = (1/3) sum_d < |u(x + l dx e_d) - u(x)|^2 >_x,  l = 1..nl (nl <= N/2), host [batch][nl]. */
int ns_structure_function(ns_solver* h, double* S_out, int nl);
/* Structure function of order p > 0 (the statistics the paper's ensembles are evaluated with, PAPER.md:L164, L309;
 * reading A15 extended): S_out[b][l-1] = (1/3) sum_d < |u(x + l dx e_d) - u(x)|^p >_x with the Euclidean norm of the
 * vector increment, evaluated in physical space on the N grid, l = 1..nl (nl <= N/2), host [batch][nl].
 * NS_ERR_INVALID_ARG for p <= 0, NULL or nl out of range.  Overwrites the library's workspaces, not the state. */
int ns_structure_function_p(ns_solver* h, double p, double* S_out, int nl);
/* Pointwise ensemble moments of the empirical measure (Algorithm 1; the mean and variance fields of
 * its Fig. 9-10): over the batch samples b = 0..batch-1 on the N grid,
 *   mean_out[c][x] = (1/batch) sum_b u_b,c(x),   var_out[c][x] = (1/batch) sum_b (u_b,c(x) - mean[c][x])^2,
 * each [3][N][N][N] reals of the solver dtype in caller memory `ms`; either pointer may be NULL (not both).
 * Overwrites the library's workspaces, not the state. */
int ns_ensemble_moments(ns_solver* h, void* mean_out, void* var_out, ns_memspace ms);

/* Simulation time of one sample; NaN if `sample` is out of range. */
double ns_time(const ns_solver* h, int sample);
/* Per-pass timing with CUDA events recorded on the solver's stream between the kernels of the RHS
 * (measurement aid for bench.py; adds one event record per kernel when enabled).  ns_profile(h, 1)
 * synchronises, clears the accumulators and enables; ns_profile(h, 0) disables.  ns_profile_read
 * synchronises and returns, for the 8 passes {a1 col_inv_x, a2 col_inv_y, a3 z_inv_prod, a4 z_fwd,
 * a5 col_fwd_y, a6 col_fwd_x, a7 spectral, other}, the accumulated milliseconds ms_out[8] and launch
 * counts count_out[8] (host arrays) since it was enabled. */
int ns_profile(ns_solver* h, int enable);
int ns_profile_read(ns_solver* h, double* ms_out, long long* count_out);
/* Number of kernels the library has launched on this handle so far (for bench.py's gpu_launches). */
long long ns_kernel_launches(const ns_solver* h);
/* Device bytes held by the handle. */
long long ns_device_bytes(const ns_solver* h);
/* Message of the last failed call on h ("" if none).  h == NULL returns the message of the last
 * failed ns_create on this thread. */
const char* ns_last_error(const ns_solver* h);

#ifdef __cplusplus
}
#endif
#endif /* NS_H_ */

/* ns2d.h -- C ABI of the TWO-DIMENSIONAL solver of libns: batched pseudo-spectral Navier-Stokes right-hand side and SSP-RK3
 * step on the periodic torus [0,2pi)^2, hand-written CUDA for one NVIDIA B200 (sm_100a).
 *
 * The paper's solver exists in a two- and a three-dimensional version (section 4: "the 2D solver is validated by
 * simulating some analytically known solutions ... the 2D Taylor-Green Vortex, or the vortex patch"; L394, section 7: "both two-
 * and three-dimensional large-scale statistical solutions").  This is the same discretisation as ns.h with d = 2: eq. (2.1)-(2.4)
 * (PAPER.md:L96-116), Algorithm 2 + eq. (2.5) (L122-136), eq. (2.6) (L146-153), with the readings A1..A20 of DESIGN.md section 3;
 * ensembles (Algorithm 1, L82-90) are the leading `batch` index -- in two dimensions typically a very large one.
 *
 * Conventions (those of ns.h unless stated)
 *   N         grid points per axis: any even N, 16 <= N <= 512.  The transforms run on the transform grid Nt = 128, 256 or 512
 *             (the smallest >= N; ns2d_transform_grid) with the padded grid M = 3 Nt / 2 >= 3N/2 (the padded size
 *             is rounded up to one the transforms are fast for); the state is truncated to the user's N and all public arrays have
 *             the user's N, exactly as in ns.h; max|u| is a maximum over the M^2 points of the padded grid in use.
 *   spectral  complex interleaved of `dtype`, shape [batch][2][N][N/2+1], index [b][component][ikx][iky], iky >= 0 fastest (r2c
 *             half spectrum along y); normalised coefficients; entries with an index == N/2 are zero (reading A3).
 *   physical  reals of `dtype`, shape [batch][2][N][N], index [b][component][ix][iy], x_j = 2 pi j / N.
 *   memspace, stream, errors, non-finite states, threads: as in ns.h (ns_params, ns_dtype, ns_memspace, ns_status are shared).
 */
#ifndef NS2D_H_
#define NS2D_H_

#include "ns.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ns2d_solver ns2d_solver; /* opaque */

/* Create a solver for `batch` independent samples on an N^2 grid; `p` may be NULL (inviscid).  One device arena of about
 * 11 * batch * N^2 * sizeof(complex) bytes (ns2d_device_bytes returns the exact figure). */
int ns2d_create(ns2d_solver** out, int N, int batch, const ns_params* p, ns_dtype dtype, void* cuda_stream);
int ns2d_destroy(ns2d_solver* h);

/* State from PHYSICAL samples [batch][2][N][N] (u(0) = P_N u_0, eq. 2.1 third line): analysis transform with 1/N^2, Nyquist
 * lines zeroed, Leray projector (eq. 2.5) for k != 0, mean kept.  Resets every sample's time to 0. */
int ns2d_set_initial(ns2d_solver* h, const void* u_phys, ns_memspace ms);
/* Set / get the state in SPECTRAL form, no projection; get -> set is bit exact; sample times unchanged. */
int ns2d_set_spectral(ns2d_solver* h, const void* u_hat, ns_memspace ms);
int ns2d_get_spectral(ns2d_solver* h, void* u_hat_out, ns_memspace ms);
/* rhs_hat_out = R(state) = (1 - k k^T/|k|^2)(-i k^T F[u (x) u]_k) - d_k u_hat_k (Algorithm 2 + eq. 2.5 + viscous term of eq. 2.1). */
int ns2d_rhs(ns2d_solver* h, void* rhs_hat_out, ns_memspace ms);

/* One SSP-RK3 step (eq. 2.6): the same dt for all samples / per-sample CFL step dt_b = min(cfl (2 pi/N)/umax_b, t_end - t_b) with
 * umax_b the maximum over the padded grid of |u|_2 evaluated on the device (reading A10) / caller-given steps.
 * Semantics of dt_out, finished samples and the replay call exactly as ns_step_cfl / ns_step_dts. */
int ns2d_step(ns2d_solver* h, double dt);
int ns2d_step_cfl(ns2d_solver* h, double cfl, double t_end, double* dt_out);
int ns2d_step_dts(ns2d_solver* h, const double* dt);
/* Integrate every sample to t_end (Algorithm 1, "evolve the sample"); as ns_advance. */
int ns2d_advance(ns2d_solver* h, double cfl, double t_end, int max_steps, int* steps_done);

/* umax_out[batch] (host): max over the padded M^2 grid of the Euclidean |u| of the current state. */
int ns2d_max_velocity(ns2d_solver* h, double* umax_out);
/* Physical velocity on the N grid, [batch][2][N][N] (the "whole flow field" writer). */
int ns2d_get_fields(ns2d_solver* h, void* u_phys_out, ns_memspace ms);
/* Ring spectra (readings A14 / A20 with d = 2), host [batch][nbins] doubles:
 *   E[b][K] = 1/2 sum_{K-1/2 <= |k| < K+1/2} |u_hat_k|^2,  Z[b][K] the same with omega_hat = i (kx u2_hat - ky u1_hat). */
int ns2d_energy_spectrum(ns2d_solver* h, double* E_out, int nbins);
int ns2d_enstrophy_spectrum(ns2d_solver* h, double* Z_out, int nbins);

double ns2d_time(const ns2d_solver* h, int sample);
/* Per-pass timing as ns_profile; the 4 passes are {b1 x inverse, b2 fused y (inverse + flux + forward), b3 x forward, b4 spectral}. */
int ns2d_profile(ns2d_solver* h, int enable);
int ns2d_profile_read(ns2d_solver* h, double* ms_out /*[4]*/, long long* count_out /*[4]*/);
int ns2d_transform_grid(const ns2d_solver* h);   /* Nt; the padded grid is 3 Nt / 2 */
long long ns2d_kernel_launches(const ns2d_solver* h);
long long ns2d_device_bytes(const ns2d_solver* h);
const char* ns2d_last_error(const ns2d_solver* h);

#ifdef __cplusplus
}
#endif
#endif /* NS2D_H_ */

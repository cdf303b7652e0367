/* ns_mg.h -- C ABI of the MULTI-DEVICE solver of libns: ONE sample of the spectral hyperviscosity Navier-Stokes right-hand side
 * and SSP-RK3 step distributed over P GPUs of one node by slab decomposition.
 *
 * The paper's topic ("the computational domain is decomposed into slabs"; section 3.1-3.3: the transforms
 * along the rank-local axes are done first, the data is transposed to make the distributed axis local, then the remaining axis
 * is transformed; Algorithm 3; the transpose moves only partially padded data).  Its design -- MPI ranks, host-staged
 * MPI_Alltoall -- is prior art; here one process drives the P devices ("cuFFT can only distribute over multiple GPUs given they
 * are managed by the same process", L177, is the model that fits one NVLink node), each device has its own stream, and the
 * transpose is FUSED into the transform pass that produces the data: the kernel stores every output row straight into the
 * memory of the device that owns it (peer stores over NVLink, overlapped with the butterflies of the next tile), ordered
 * between the devices' streams by events: no separate transpose pass, no host staging, no host synchronisation inside a step.
 *
 * Decomposition (P devices, rank r = position in the device list; Nyl = N/P, Ml = M/P, M = 3N/2):
 *   spectral side   rank r owns the ky rows [r Nyl, (r+1) Nyl) of every array [comp][kx][ky][kz]: a1 (inverse x pass), a6 (forward
 *                   x pass), a7 (spectral / RK kernel) and the state live here;
 *   physical side   rank r owns the px planes [r Ml, (r+1) Ml) of [comp][px][ky][kz]: a2 (y pass), a3+a4 (fused z kernel: padded
 *                   physical data never leaves the SM) and a5 run here;
 *   exchange A      inside a1: block (px in slab s, ky in slab r) of 3 components is stored by rank r into rank s   (3 M N H / P^2 per pair)
 *   exchange B      inside a5: block (px in slab r, ky in slab s) of the 5 trace-free flux components goes back     (5 M N H / P^2 per pair)
 * The kernels are the ones of ns.h (same launchers, sub-ranges by pointer / stride); max|u| for the CFL step is reduced over the
 * devices by peer copies of P scalars.  Results equal those of ns.h on one device to round-off (the arithmetic per line is
 * identical; only the order of the max reduction differs, which is exact).
 *
 * Conventions: those of ns.h (layouts, normalisation, Nyquist planes, ns_params, ns_dtype, ns_status).  Restrictions: batch = 1;
 * N a transform grid of ns.h (p 2^a, p in {1, 3, 5, 7, 15}, 32 <= N <= 640, N/2 a multiple of 8, fp32: 16) with N and 3N/2
 * divisible by P; a decomposition whose slabs the pass kernels cannot tile is rejected by ns_mg_create; the state is set and
 * read in SPECTRAL form in host memory (physical-space entry points stay with ns.h).  The device list may name the same device
 * more than once: the P ranks then share that GPU, which is how the decomposition is tested on a single-GPU machine.
 */
#ifndef NS_MG_H_
#define NS_MG_H_

#include "ns.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ns_mg_solver ns_mg_solver; /* opaque */

/* Create a solver for one sample on an N^3 grid over the P devices devices[0..P-1] (CUDA device ordinals; repeats allowed).
 * Enables peer access between distinct devices (NS_ERR_CUDA if a pair cannot access each other).  Each rank allocates about
 * 24 N^3 sizeof(complex) / P bytes.  `p` may be NULL (inviscid). */
int ns_mg_create(ns_mg_solver** out, int N, int P, const int* devices, const ns_params* p, ns_dtype dtype);
int ns_mg_destroy(ns_mg_solver* h);

/* State in spectral form, host memory, public layout [3][N][N][N/2+1] of ns.h; get -> set is bit exact.  Synchronous. */
int ns_mg_set_spectral(ns_mg_solver* h, const void* u_hat_host);
int ns_mg_get_spectral(ns_mg_solver* h, void* u_hat_host);
/* rhs_hat_host = R(state), the right-hand side of ns_rhs (Algorithm 2 + eq. 2.5 + viscous term of eq. 2.1).  Synchronous. */
int ns_mg_rhs(ns_mg_solver* h, void* rhs_hat_host);
/* One SSP-RK3 step (eq. 2.6) with the given dt / with dt = min(cfl (2 pi/N)/umax, t_end - t), umax the maximum of |u| over the
 * padded grid of all devices (reading A10); *dt_out (may be NULL) receives the step taken (then the call synchronises). */
int ns_mg_step(ns_mg_solver* h, double dt);
int ns_mg_step_cfl(ns_mg_solver* h, double cfl, double t_end, double* dt_out);
/* max over the padded grid of the Euclidean |u| of the state (host scalar). */
int ns_mg_max_velocity(ns_mg_solver* h, double* umax_out);

double ns_mg_time(const ns_mg_solver* h);
/* Bytes one exchange A + one exchange B move between DIFFERENT ranks per RHS evaluation (the slab transpose volume). */
long long ns_mg_exchange_bytes(const ns_mg_solver* h);
long long ns_mg_kernel_launches(const ns_mg_solver* h);
long long ns_mg_device_bytes(const ns_mg_solver* h);   /* per rank */
const char* ns_mg_last_error(const ns_mg_solver* h);

#ifdef __cplusplus
}
#endif
#endif /* NS_MG_H_ */

/* ns_noalloc.h -- ONE entry point of libns that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid allocation).
 *
 * ns_noalloc_energy_spectrum: the shell-averaged energy spectrum of ns_energy_spectrum (reading A14 of DESIGN.md:
 * E[b][K] = 1/2 sum over K-1/2 <= |k| < K+1/2 of |u_hat_k|^2, full-spectrum weights, Nyquist planes excluded) of a spectral state the
 * CALLER holds in device memory, without a solver handle.  The bins are accumulated with atomics in a scratch array that is a
 * file-scope `static __device__` array inside the library (NS_NOALLOC_MAX_VALUES doubles = 128 KiB, resident on every GPU that loads
 * libns from load until exit); its device address is resolved once per device with cudaGetSymbolAddress.  The call performs no
 * cudaMalloc / cudaFree and calls no allocating library routine: three kernel launches on the caller's stream (clear, accumulate,
 * copy out) and, for a host output, one cudaMemcpyAsync + cudaStreamSynchronize.
 *
 *   u_hat_dev   DEVICE pointer, complex interleaved of `dtype`, the public spectral layout of ns.h: [batch][3][N][N][N/2+1]
 *   N           grid points per axis: even, 2 <= N <= 4096 (no transform is involved, so any even N)
 *   nbins       1 <= nbins <= 4096, and batch * nbins <= NS_NOALLOC_MAX_VALUES -- larger requests are rejected with
 *               NS_ERR_INVALID_ARG (nothing is truncated); modes with |k| + 1/2 >= nbins are dropped, as in ns_energy_spectrum
 *   E_out       [batch][nbins] doubles in caller memory tagged by `out_ms` (NS_DEVICE: written by the last kernel, the call is
 *               asynchronous on the stream; NS_HOST: copied, the call synchronises the stream)
 *   cuda_stream a cudaStream_t cast to void* (NULL = the legacy default stream); the device current at the call is used
 *   errbuf      optional: receives the error text on failure (errbuf_len bytes including the terminator); may be NULL
 * Returns NS_OK or a negative ns_status (ns.h).
 *
 * SHARED SCRATCH: every call on a device uses the same array, which keeps the contents of the last call; the entry point clears the
 * part it uses first.  Calls that OVERLAP on the GPU (two streams, two host threads) race on it: serialise them.  The first call on
 * a device resolves the symbol address (a one-time set-up step that may load the module): make it once before starting a graph
 * capture.  The existing entry points of ns.h are unchanged and do not use this array.
 */
#ifndef NS_NOALLOC_H_
#define NS_NOALLOC_H_

#include "ns.h"

#ifdef __cplusplus
extern "C" {
#endif

#define NS_NOALLOC_MAX_VALUES 16384 /* doubles of scratch = the largest batch * nbins */

int ns_noalloc_energy_spectrum(const void* u_hat_dev, int N, int batch, ns_dtype dtype, int nbins, double* E_out, ns_memspace out_ms,
                               void* cuda_stream, char* errbuf, int errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* NS_NOALLOC_H_ */

/* sparse_sv_static.h -- the ONE entry point of libsparse_sv.so that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  Every call of include/sparse_sv.h works on a handle whose arena was allocated at sv_create; this call
 * needs no handle.  It computes the mass of a term array (Eq. 4: sum over the terms of |a|^2 -- the quantity
 * the renormalisation of PAPER.md:96 divides by) with the same two kernels' arithmetic as
 * sv_norm: a fixed grid of partial sums, then one block that adds the partials, every addition rounded separately
 * and in a fixed order (D1), so the result is the same bits on every run and the same bits as sv_norm on
 * the same amplitude array.
 *
 * Scratch: the partial sums live in a file-scope `static __device__` array of SV_NORM_STATIC_SCRATCH_BYTES bytes
 * inside the library (csrc/sv_static.cu).  Every GPU that loads the library holds those bytes until the process
 * exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *
 * ALL calls on one device share that array, and it keeps the last call's contents.  Nothing in it has to start at
 * zero (every partial a call reads was written by that call first), so there is nothing to clear; but two calls
 * that OVERLAP on the GPU (different streams, no dependency between them) race on it and both results are
 * undefined.  Calls on one stream, or ordered by events, are safe.  Different devices have different copies.
 */
#ifndef SPARSE_SV_STATIC_H
#define SPARSE_SV_STATIC_H

#include "sparse_sv.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Size of the static scratch array: 1024 partial sums of 8 bytes. */
#define SV_NORM_STATIC_SCRATCH_BYTES 8192
/* Largest n the call accepts: 2^32 terms (64 GiB of amplitudes). */
#define SV_NORM_STATIC_MAX_TERMS (1ull << 32)

/* *dev_mass = sum_{i<n} re_i^2 + im_i^2.
 *   dev_amps  DEVICE pointer, n complex128 amplitudes (16-byte aligned), read only; caller-owned.  May be NULL if n == 0.
 *   n         number of terms, 0 <= n <= SV_NORM_STATIC_MAX_TERMS; n == 0 gives 0.0.
 *   dev_mass  DEVICE pointer to one double (8-byte aligned), written by the call; caller-owned.
 *   stream    a cudaStream_t passed as void* (NULL = the legacy default stream) of the CURRENT device; the two kernels
 *             are enqueued on it and the call returns without synchronising: read *dev_mass after the stream has
 *             reached that point.
 * Returns SV_OK; SV_ERR_INVALID_ARG for a null / misaligned pointer, a pointer that CUDA reports as plain host memory,
 * or n > SV_NORM_STATIC_MAX_TERMS (nothing is enqueued); SV_ERR_CUDA if the address of the scratch array cannot be
 * obtained or a launch fails.  sv_static_last_error() names the reason.
 * The first call on a device looks up the device address of the scratch array (cudaGetSymbolAddress; no allocation by
 * this library, but the CUDA runtime may load the module then): make that first call outside a graph capture, or call
 * sv_norm_static_init() there. */
int sv_norm_static(const sv_c128 *dev_amps, uint64_t n, double *dev_mass, void *stream);

/* Set-up of the current device for sv_norm_static (idempotent, thread safe; sv_norm_static calls it itself).
 * Returns SV_OK or SV_ERR_CUDA.  No device work. */
int sv_norm_static_init(void);

/* Reason of the last error sv_norm_static / sv_norm_static_init returned on THIS thread ("" if none); a static string
 * or a thread-local buffer owned by the library, valid until the thread's next call. */
const char *sv_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SPARSE_SV_STATIC_H */

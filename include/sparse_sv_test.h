/* sparse_sv_test.h -- TEST HOOKS of libsparse_sv.so; not part of the product API (include/sparse_sv.h).
 *
 * The fused call sv_apply_gate_truncate (apply, then truncate) estimates a floor for the cut that
 * follows from a sample of the gate's outputs, with a statistical safety margin, and re-runs the pass without a
 * floor when the margin turns out to have failed.  That re-run path is
 * practically unreachable with the real margin; this hook lets a test reach it.
 */
#ifndef SPARSE_SV_TEST_H
#define SPARSE_SV_TEST_H

#include "sparse_sv.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Sample points added to the margin of the output floor (default 0).  A negative value makes the margin fail, so
 * that the pass stores fewer than max_terms outputs and is re-run without a floor (sv_stats.fallbacks counts it).
 * s: handle (host pointer).  Returns SV_OK, or SV_ERR_INVALID_ARG for a null handle.  No device work. */
int sv_test_set_pre_slack(sv_state *s, long long slack);

/* Diagnostic: bit q of *mask (host pointer) is set iff qubit q has the same value in every term of the state (a pending
 * truncation is taken into account).  One pass over the state (24 B per term), synchronises the state's stream.
 * Returns SV_OK, SV_ERR_INVALID_ARG (null pointer) or SV_ERR_CUDA. */
int sv_test_definite_qubits(sv_state *s, uint64_t *mask);

#ifdef __cplusplus
}
#endif
#endif /* SPARSE_SV_TEST_H */

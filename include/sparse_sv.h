/* sparse_sv.h -- C ABI of the B200-native sparse, truncated state-vector gate engine.
 *
 * Method: arxiv/paper_2607_07816 "A Sparse and Truncated State Vector Simulator for
 * Peaked Circuits".  A state is stored only as its nonzero terms, each a
 * (uint64 basis index, complex128 amplitude) pair.  All state
 * arrays live in device memory for the whole simulation; only results cross to the
 * host.
 *
 * Conventions:
 *   - qubit q is bit q of the 64-bit key (LSB = qubit 0), 1 <= n_qubits <= 64;
 *   - a gate matrix U is HOST memory, row-major 2^m x 2^m, U[r * 2^m + c]; bit j of the
 *     local index r / c is the key's bit qubits[j]; 1 <= m <= 4;
 *   - "probability" p = re*re + im*im in fp64; the total order used for truncation and
 *     readout is (p descending, key ascending).
 *
 * Every pointer below is a HOST pointer unless it says DEVICE.  The handle owns all
 * device memory it allocates; caller buffers are only read or written during the call
 * and never freed.  No C++ exception crosses this boundary.  Return value: SV_OK or a
 * negative error; on any error the logical state is unchanged (gates are applied out of
 * place and committed by swapping buffers).  Work is enqueued on the state's CUDA
 * stream; calls that return a value to the host synchronise that stream.
 */
#ifndef SPARSE_SV_H
#define SPARSE_SV_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sv_state sv_state;              /* opaque */
typedef struct { double re, im; } sv_c128;     /* = C99 double _Complex layout */

enum {
    SV_OK = 0,
    SV_ERR_INVALID_ARG = -1,
    SV_ERR_CAPACITY = -2,  /* a gate's output (before truncation) would exceed `capacity` */
    SV_ERR_NOMEM = -3,
    SV_ERR_CUDA = -4
};

/* gate classes reported by sv_get_stats */
enum { SV_CLASS_NONE = 0, SV_CLASS_DIAGONAL = 1, SV_CLASS_XOR = 2, SV_CLASS_GROUP = 3 };

typedef struct {
    int      gate_class;   /* SV_CLASS_* of the last sv_apply_gate                          */
    int      m;            /* its number of qubits                                          */
    int      active_bits;  /* qubits on which U is not block diagonal (0 for diagonal)      */
    int      passes;       /* full passes over the state the call made                      */
    uint64_t n_in;         /* terms before the last call                                    */
    uint64_t n_out;        /* terms after it (N_pre for a gate, N_kept for a truncate)      */
    uint64_t launches;     /* kernels launched by this handle since creation                */
    uint64_t fallbacks;    /* sampled estimates that missed: truncations that re-ran the full select, fused gates that re-ran without a floor */
    uint64_t n_mid;        /* sv_apply_gate_truncate: terms of the gate's output before the cut (logical; not all were written) */
    uint64_t pre_dropped;  /* outputs the last gate did not write because the cut that follows drops them (fused call)          */
    uint64_t small_gates;  /* gates sv_apply_circuit has run through its single-block path since creation                       */
} sv_stats;

/* Bytes of device memory a state of this capacity needs (for sv_create_in_arena). */
size_t sv_arena_bytes(uint64_t capacity);

/* New state |0...0>: one term, key 0, amplitude 1+0i.  `capacity` is the
 * largest number of terms that may exist at any instant, including a gate's output
 * before truncation.  Allocates with cudaMalloc on the current device, uses its own
 * stream. */
int sv_create(int n_qubits, uint64_t capacity, sv_state **out);

/* Same, inside caller-owned DEVICE memory (e.g. a torch uint8 tensor) of at least
 * sv_arena_bytes(capacity) bytes, 256-byte aligned, on `cuda_stream` (a cudaStream_t;
 * NULL = the legacy default stream).  The arena must outlive the handle. */
int sv_create_in_arena(int n_qubits, uint64_t capacity, void *dev_arena, size_t arena_bytes,
                       void *cuda_stream, sv_state **out);

void sv_destroy(sv_state *s);

/* Apply the m-qubit gate U to `qubits` (distinct, each < n_qubits): every tuple of 2^m
 * amplitudes whose basis states differ only in those qubits is multiplied by U, the
 * contributions to one basis state are summed in ascending local column index with
 * separately rounded multiplies and adds, and results that are exactly 0+0i are dropped
 * (PAPER.md:47, :110-120).  U is not checked for unitarity.  Asynchronous except for a
 * term-count read-back when the gate can change the number of terms. */
int sv_apply_gate(sv_state *s, const int *qubits, int m, const sv_c128 *U);

/* Truncate: keep the smallest prefix, in (p desc, key asc)
 * order, whose mass is >= min_mass * (current total mass); then at most max_terms of it;
 * then multiply the kept amplitudes by 1/sqrt(kept mass).  max_terms == 0: no cap.
 * min_mass >= 1: no mass threshold; min_mass <= 0 or NaN: SV_ERR_INVALID_ARG.  At least
 * one term is kept.  If nothing is dropped the state is left bitwise untouched.
 * *kept_fraction (nullable) receives kept mass / total mass. */
int sv_truncate(sv_state *s, uint64_t max_terms, double min_mass, double *kept_fraction);

/* sv_apply_gate followed by sv_truncate with these arguments, as ONE call (every
 * gate, or fused block of gates, is applied and the state truncated before the next).  The result
 * -- kept set, amplitudes, *kept_fraction -- is that of the two calls; knowing the cut that
 * follows, the engine may estimate a floor for it from a sample of the gate's outputs and never
 * write the outputs below that floor: less memory traffic,
 * and a peak term count near max_terms instead of 2^m x N_in.  Arguments, errors and ownership as
 * for the two calls; on an error from the gate nothing changed, on an error from the truncation
 * the gate has been applied.  sv_get_stats then reports the gate's class, n_in = terms before the
 * gate, n_out = terms kept. */
int sv_apply_gate_truncate(sv_state *s, const int *qubits, int m, const sv_c128 *U,
                           uint64_t max_terms, double min_mass, double *kept_fraction);

/* A sequence of gates, each followed by the same truncation ("for each block ... apply ... truncate"), as ONE
 * call: gate g has gate_m[g] qubits; qubit lists and row-major 2^m x 2^m matrices are concatenated in gate_qubits / gate_U
 * (conventions of sv_apply_gate; fused blocks from sv_fuse_gates can be passed as they are).  The result is that of
 * n_gates calls of sv_apply_gate_truncate(.., max_terms, min_mass, ..); kept_fractions (nullable, n_gates doubles) receives
 * each step's kept mass / mass before.  Knowing the gates ahead, the engine does not return to the host between steps when
 * it need not: while the state has at most 4096 terms and a gate's output fits 4096 entries, every step is one
 * single-block kernel (gate + zero drop + cut + renormalisation in shared memory, the term count kept on the device) and a
 * batch of up to 64 steps costs one synchronisation -- the regime the paper reports after reordering and fusion
 * (< 2^5 terms; "a fixed overhead ... at low values of k").  Larger states take the streaming passes
 * gate by gate.  The two paths agree up to the rounding of the mass sums (fp64 tree sums in the single-block kernel, exact
 * integer sums in the streaming path): a cut can differ only at a knife edge (R22).  *n_done (nullable) receives
 * the number of gates applied: n_gates on SV_OK; on an error the state is that after *n_done gates.  The whole list is
 * validated first (SV_ERR_INVALID_ARG then changes nothing).  Synchronises the stream. */
int sv_apply_circuit(sv_state *s, int n_gates, const int *gate_m, const int *gate_qubits, const sv_c128 *gate_U,
                     uint64_t max_terms, double min_mass, double *kept_fractions, int *n_done);

/* Gate fusion ("for each block of single- and two-qubit gates we fuse those gates into a
 * multi-qubit unitary operation", one state update and one truncation per block).  HOST ONLY: no device work.
 * The n_gates input gates -- gate_m[g] qubits each, their qubit lists concatenated in gate_qubits, their row-major
 * 2^m x 2^m matrices concatenated in gate_U (conventions of sv_apply_gate) -- are merged, in order and greedily,
 * into blocks: a gate joins the running block while the union of qubits has at most max_m (<= SV_FUSE_MAX_M)
 * members, else the block is closed and the gate opens the next one.  A block's qubits are listed in order of first
 * appearance (local bit j = j-th listed qubit); its matrix is the product of its gates, later gates on the left.
 * Outputs (caller-owned): *n_blocks; block_m[n_gates]; block_qubits[sum of gate_m], concatenated; block_U,
 * concatenated, block_U_capacity entries available (n_gates * 4^max_m always suffices).  Each block is a gate for
 * sv_apply_gate / sv_apply_gate_truncate.  SV_ERR_INVALID_ARG: bad sizes, a repeated or out-of-range qubit, a gate
 * wider than max_m, or not enough room in block_U. */
#define SV_FUSE_MAX_M 4
int sv_fuse_gates(int n_gates, const int *gate_m, const int *gate_qubits, const sv_c128 *gate_U, int max_m,
                  int *n_blocks, int *block_m, int *block_qubits, sv_c128 *block_U, size_t block_U_capacity);

/* Gate reordering ("we reorder the gates so that, during simulation, the set of currently active
 * qubits is kept as small as possible, while the introduction of additional qubits is postponed for as long as the
 * circuit dependencies allow ... we only reorder commuting gates or dependency-compatible gates").  HOST ONLY: no
 * device work.  The paper states the goal, not an algorithm; the reading (R20) is a greedy list schedule.
 * Two gates conflict when they share a qubit, unless both are flagged in gate_diag (nullable; gate_diag[g] != 0: U of
 * gate g is diagonal, and diagonal gates commute).  A gate is ready once every EARLIER gate it conflicts with has been
 * scheduled, so every conflicting pair keeps its order and the reordered list is the same operator.  A qubit is
 * active once a scheduled gate has touched it.  Every step schedules the ready gate that activates the fewest new
 * qubits, ties to the lowest original index.  gate_m / gate_qubits as for sv_fuse_gates (qubits < 64, distinct within
 * a gate, any m <= 64: matrices are not needed).  Outputs (caller-owned, n_gates entries each): order[t] = index of
 * the gate scheduled t-th; n_active_after[t] (nullable) = active qubits after it.  SV_ERR_INVALID_ARG: bad sizes, a
 * repeated or out-of-range qubit. */
int sv_reorder_gates(int n_gates, const int *gate_m, const int *gate_qubits, const unsigned char *gate_diag,
                     int *order, int *n_active_after);

/* *mass = sum of |a|^2 over all terms (Eq. 4) -- the mass, not its root. */
int sv_norm(sv_state *s, double *mass);

/* The min(k, count) most probable terms, sorted by (p desc, key asc) (PAPER.md:61,
 * :132-134).  keys / amps / probs are caller-owned host arrays of k entries; any may be
 * NULL.  *n_written (nullable) receives the number of records written. */
int sv_top(sv_state *s, uint64_t k, uint64_t *keys, sv_c128 *amps, double *probs,
           uint64_t *n_written);

/* Current number of stored terms. */
int sv_num_terms(sv_state *s, uint64_t *n);

/* Replace the state by n host terms (test / checkpoint hook).  Keys must be distinct
 * and < 2^n_qubits, amplitudes nonzero, n <= capacity; else SV_ERR_INVALID_ARG. */
int sv_load(sv_state *s, const uint64_t *keys, const sv_c128 *amps, uint64_t n);

/* Same with DEVICE source arrays (no host copy; used to time device-resident input). */
int sv_load_device(sv_state *s, const uint64_t *dev_keys, const sv_c128 *dev_amps, uint64_t n);

/* Tuning knob.  SV_OPT_SAMPLE_MIN_TERMS: states with at least this many terms find the
 * truncation cut with the sampled one-pass path (sv_sample_select.cu; default 2^21), smaller
 * ones with the full-state radix select.  Both are exact; tests force either.  The same threshold gates the
 * output floor of sv_apply_gate_truncate. */
enum { SV_OPT_SAMPLE_MIN_TERMS = 0, SV_OPT_SMALL_STATE_PATH = 2,   /* 2: 1 (default) / 0: sv_apply_circuit may / may not use its single-block path */
       SV_OPT_TWO_BIT_PASS = 3 };   /* the final pass of a dense multi-qubit gate (every entry of U nonzero) brings its last TWO missing qubits to
                                     * the low bit positions at once -- one pass over the state less --: 0 never (one pass per missing qubit),
                                     * 1 for every such gate applied through sv_apply_gate, 2 (default) for those on three or four mixing
                                     * qubits, where it is measured faster.  sv_apply_gate_truncate and sv_apply_circuit never use it.
                                     * The result is the same bit for bit. */
int sv_set_option(sv_state *s, int option, uint64_t value);

/* Statistics of the last call and the launch counter. */
int sv_get_stats(sv_state *s, sv_stats *out);

/* Optional per-kernel timing.  sv_profile(s, 1) resets the counters and makes every later
 * launch of the main kernels be bracketed by CUDA events on the state's stream;
 * sv_profile_get synchronises and returns, for one kernel, the summed device time, the
 * number of launches and the ALGORITHMIC bytes they had to move (DESIGN.md "Kernels":
 * diagonal 40 B/term; bit move 48 B/term; final pass of a one-bit gate (bitpass: monomial blocks,
 * position preserving; bitpass_gen: general blocks) and of a multi-bit gate (grouppass) 24 B x (N_in + N_out); select histogram 16 B/term; compaction
 * 24 B x (N_in + N_kept); sampled classification 16 B/term). */
enum { SV_K_DIAG = 0, SV_K_MOVE = 1, SV_K_BITPASS = 2, SV_K_SELHIST = 3, SV_K_COMPACT = 4, SV_K_CLASSIFY = 5, SV_K_GROUPPASS = 6, SV_K_BITPASS_GEN = 7, SV_K_COUNT = 8 };
typedef struct { double ms; uint64_t launches; double alg_bytes; } sv_kernel_prof;
int sv_profile(sv_state *s, int enable);
int sv_profile_get(sv_state *s, int kernel, sv_kernel_prof *out);

/* Device-side structural check (tests): keys strictly ascending in the engine's storage
 * order, all below 2^n_qubits, no stored exact zero.  *ok = 1 if all hold. */
int sv_check_invariants(sv_state *s, int *ok);

/* Last error message of this handle ("" if none); valid until the next call on it. */
const char *sv_last_error(const sv_state *s);

/* Block until all work enqueued on the state's stream has finished. */
int sv_sync(sv_state *s);

#ifdef __cplusplus
}
#endif
#endif /* SPARSE_SV_H */

// Internal declarations shared by the engine's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

typedef unsigned long long u64;
typedef unsigned int u32;

#define SV_MAX_M 4
#define SV_THREADS 256
#define SV_SEL_BINS 4096        // 12-bit digits for the radix select

// Gate tables in device memory, in PHYSICAL pattern indexing.
struct GateTab {
    int ma;                 // active bits: they sit at physical positions 0..ma-1 when the group kernel runs
    int mc;                 // control-like bits
    int ctrl_pos[SV_MAX_M]; // physical position of control bit i (layout after the final move)
    int colorder[16];       // colorder[t] = physical active pattern of the t-th logical column
    double2 U[256];         // U[((cx << ma | xr) << ma) | xc]
};

// One tile boundary of a bit-move pass: a merge-path split inside one block (= maximal
// range of keys that agree above the moved bit).  A = keys with the bit 0, B = bit 1.
struct TileDesc {
    u64 ia;   // first A element not yet consumed (global index)
    u64 ib;   // first B element not yet consumed
    u64 mid;  // start of the block's B run
    u64 e;    // end of the block
};

// One tile boundary of a TWO-bit pass (bits pH > pL go to the two least-significant positions in one pass; sv_gate.cu
// find_splits2, sv_dense.cu).  With the stored key read as (high, bH, mid, bL, low) and rest = (high, mid, low), the
// boundary is a value R = (h, m, l) of rest; the entries with rest < R are the stored ranges
//   [0, p00)  [m2a, p01)  [m1, p10)  [m2b, p11)
// p00 / p01 / p10 / p11: lower bounds of (h, bH, m, bL, l) for the four patterns of (bH, bL); m1: start of the bH = 1
// half of block h; m2a / m2b: start of the bL = 1 run of the sub-block (h, bH, m) of either half.
struct TileDesc2 {
    u64 p00, m2a, p01, m1, p10, m2b, p11, pad_;
};
// ... and the tile between two boundaries as contiguous pieces of the input (make_pieces2 in sv_gate.cu): the table
// follows the ntiles + 1 boundaries in the descriptor area; per tile the start indices of pieces 0 .. 7, then their
// lengths, 32 bits each (0: no piece; the pieces are in stored order and not empty).
#define SV_PIECES2 8
#define SV_PIECES2_WORDS 12

// Radix-select state (device resident; one per handle).  See sv_radix_select.cu.
struct SelState {
    int phase;           // 0 exponent level, 1 adaptive pattern levels, 2 tie keys to be extracted, 3 key levels
    int done;            // 1: PT/KT final; 2: internal inconsistency
    int count_active, mass_active;
    int E, pad_;         // exponent field shared by the candidates (mass scale)
    u64 rmask, rval;     // resolved bits of the cutoff probability pattern
    u64 dmask;           // bit positions forming the next pattern digit
    u64 krmask, krval, kdmask;          // the same for the logical key among tied terms
    u64 k_rem;           // terms still to take from the candidates (count criterion / ties)
    double mass_rem_hi, mass_rem_lo;    // mass still to collect (mass criterion), double-double
    u64 kept_count;      // terms certainly kept so far
    double kept_hi, kept_lo;            // their mass, double-double
    double total_hi, total_lo;          // total mass S
    double min_mass;
    u64 cand_count;      // size of the current candidate bin
    u64 tie_total;       // terms with pattern == PT when the cut falls among ties
    u64 PT, KT;          // final predicate: keep iff pat > PT || (pat == PT && (KT == ~0 || lkey <= KT))
    double kept_mass, total_mass, scale, kept_fraction;
    u64 final_count;     // number of terms the predicate keeps
    u64 n_total;
    int seeded, pad2_;   // 1: the select runs on the candidates of the sampled fast path (sv_sample_select.cu)
    u64 P_lo;            // seeded: every term outside the candidates and not above them has a pattern < P_lo
    u64 below_cnt;       // seeded: terms certainly below the candidates; a cut that would need them is a band miss (done = 3)
    double pre_hi, pre_lo;   // mass of the outputs a fused apply+truncate never wrote (PreCut); part of S
};

// Sampled fast path of the truncation cut (sv_sample_select.cu): pivots and the results of the
// classification pass.  tot / abv: 128-bit fixed-point masses (low word, high word) in units of
// 2^(Eref - 1075 - 41).
struct SampleCtl {
    u64 P_hi, P_lo;      // above iff pattern > P_hi; below iff pattern < P_lo; else candidate
    int Eref, pad_;
    u64 above_cnt, below_cnt, cand_cnt, overflow;
    u64 tot[2], abv[2];
};

// Fused apply + truncate (sv_presample.cu): outputs of the gate whose probability pattern is below
// P_floor are not written by the pass; cnt / mass (double-double) describe what was left out.
struct PreCut {
    u64 P_floor;
    u64 cnt;
    double mass_hi, mass_lo;
};

// Small-state path (sv_small.cu): one thread block per gate, count on the device.
#define SV_SMALL_CAP 4096
struct SmallGate {
    int m, xm;              // qubits; the lazy X mask restricted to them (stored local pattern = true pattern ^ xm)
    int pos[SV_MAX_M];      // physical bit positions of the gate's qubits
    double2 U[256];         // 2^m x 2^m, row-major in TRUE local indices, as the caller gave it
};
struct SmallCtl {
    u64 count, n_pre;       // terms now; terms after the last gate before its cut
    int status;             // 1: a gate's input or output did not fit -- the state is that before gate fail_gate
    int fail_gate, done_gates, pad_;
};

// stored (physical) key -> logical key.  The map is a bit permutation plus the lazy X mask,
// hence linear over GF(2): logical = XOR over the 8 bytes b of lut[b * 256 + byte_b(stored)]
// (the mask is folded into table 0).  lut: DEVICE memory, 8 x 256 u64, built by the host.
struct KeyMap {
    const u64* lut;
};

// A truncation whose compaction has been deferred to the next reader of the state: a term
// survives iff pat > PT || (pat == PT && (KT == ~0 || logical key <= KT)); survivors are
// multiplied by `scale`.  active == 0: nothing pending.
struct PendPred {
    int active;
    u64 PT, KT;
    double scale;
    KeyMap km;
};

#define SV_MAX_DEV 64
int sv_cur_device(); // ordinal of the current device, clamped to SV_MAX_DEV - 1 (index of the per-device caches)
int sv_sm_count();   // SMs of the current device (cached per device)
// In place: monomial one-bit gate whose active bit is the physical LSB (partners are neighbours); applies a pending cut.
int svk_perm_lsb(u64* keys, double2* amps, u64 n, const GateTab* tab, const PendPred& pend, cudaStream_t st);
size_t svk_small_smem();
int svk_small_gates(u64* keys, double2* amps, SmallCtl* ctl, const SmallGate* gates, int n_gates, KeyMap km, u64 max_terms, double min_mass,
                    double* kept_out, u64 cap, int threads, cudaStream_t st);
int svk_count_live(const double2* amps, u64 n, u64* d_count, cudaStream_t st);
// out[0] = OR, out[1] = AND of the stored keys of the live entries (amps == nullptr: of all stored entries)
int svk_key_masks(const u64* keys, const double2* amps, u64 n, const PendPred& pd, int with_pend, u64* out, cudaStream_t st);

// ---- launchers (each enqueues on `st` and returns the number of kernels launched) ----
int svk_diag(const u64* keys, double2* amps, u64 n, const GateTab* tab, cudaStream_t st);

// Final pass of a gate with ma >= 2 active bits (sv_group.cu).  p < 0: the active bits already sit at the
// LSBs.  A pending truncation is applied while loading.  d_count[0] = stored outputs, d_count[1] = dead ones.
// pre != nullptr (fused apply + truncate): outputs below pre->P_floor (and exact zeros) are left out, see svk_bitpass.
int svk_grouppass(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int ma,
                  const GateTab* tab, const PendPred& pend, TileDesc* desc, u64* status, u64* d_count,
                  u64 cap, cudaStream_t st, cudaEvent_t e0 = nullptr, cudaEvent_t e1 = nullptr,
                  const PreCut* pre = nullptr, double* pre_mass = nullptr, u64* pre_cnt = nullptr, u32* pre_parts = nullptr,
                  int dense = 0, int maybe_dead = 1,    // dense: U has no zero entry and no control-like bit (sv_dense.cu)
                  int p2 = -1);                         // dense only: a SECOND bit (p2 < p) moved by the same pass, see TileDesc2

// Lean single-bit pass (sv_pair.cu): moves physical bit p to the LSB in one streaming pass.
// pair != 0: final pass of a gate with ONE active bit (tuple mat-vec + zero drop fused);
// pair == 0: pure move.  A pending truncation is applied while loading.  Writes the output
// count to *d_count.
// pre != nullptr (pair == 1 only): outputs below pre->P_floor are left out; their per-block masses and counts go
// to pre_mass / pre_cnt[0 .. *pre_parts).
int svk_bitpass(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int pair, int fixed,
                const GateTab* tab, const PendPred& pend, TileDesc* desc, u64* status, u32* tile_counter,
                u64* d_count, u64 cap, cudaStream_t st, cudaEvent_t e0 = nullptr, cudaEvent_t e1 = nullptr,
                const PreCut* pre = nullptr, double* pre_mass = nullptr, u64* pre_cnt = nullptr, u32* pre_parts = nullptr,
                u32 tnom = 0);   // tnom: nominal inputs per tile (0: the default, BP_TILE - 2)
// fused apply + truncate: pre-sample of a one-bit gate's outputs -> (sort) -> floor; per-block partials -> totals (d_count[2] = count)
int svk_pre_sample1(const u64* keys, const double2* amps, u64 n, int p, const GateTab* tab, const PendPred& pend, u32 M, u64* smp,
                    cudaStream_t st);
int svk_pre_sample_group(const u64* keys, const double2* amps, u64 n, int p, int ma, const GateTab* tab, const PendPred& pend, u32 M,
                         u64* smp, cudaStream_t st, int p2 = -1);
int svk_pre_pivot(const u64* smp_sorted, u32 M, u64 n, u32 mult, u64 max_terms, long long slack, PreCut* pre, cudaStream_t st);
int svk_pre_finish(const double* part_mass, const u64* part_cnt, u32 nparts, PreCut* pre, u64* d_count, cudaStream_t st);
int svk_find_splits(const u64* keys, u64 n, int p, int w, u32 tnom, u32 ntiles, TileDesc* desc, cudaStream_t st);
// boundaries of a two-bit pass: bits pH > pL; w low bits of the key belong to the tuple (boundaries are aligned to it);
// desc[0 .. ntiles] and, behind them, the piece table of the ntiles tiles
int svk_find_splits2(const u64* keys, u64 n, int pH, int pL, int w, u32 tnom, u32 ntiles, TileDesc2* desc, cudaStream_t st);
// Diagonal gate fused with a pending truncation (out of place, compacting).
int svk_diag_compact(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, const GateTab* tab,
                     const PendPred& pend, u64* status, u32* tile_counter, u64* d_count, cudaStream_t st);

// In-place: pending truncation (+ diagonal phases when has_phase) -> dropped terms become dead entries.
int svk_diag_pend(const u64* keys, double2* amps, u64 n, const GateTab* tab, int has_phase, const PendPred& pend, cudaStream_t st);

int svk_norm(const double2* amps, u64 n, double* partials, double* d_out, cudaStream_t st);

int svk_sel_init(SelState* ss, u64* hist, u64 n_live, u64 max_terms, double min_mass, cudaStream_t st, const PreCut* pre = nullptr);
int svk_sel_pass(int mode, const double2* amps, const u64* lkeys, u64 n, const SelState* ss, u64* hist, cudaStream_t st);
int svk_sel_extract(const u64* keys, const double2* amps, u64 n, const SelState* ss, KeyMap km, u64* lk_out, u64* hist,
                    cudaStream_t st);
int svk_sel_step(SelState* ss, u64* hist, cudaStream_t st, int expected_phase = -1);
// sampled fast path: sample -> (sort) -> pivots -> classify -> seed the select state
// xf_tab != nullptr (fused diagonal gate + truncate): the diagonal gate in xf_tab and the pending cut *pd are applied on the fly
// (sample) / in place through amps_rw (classify) before the amplitude is looked at.
int svk_ss_sample(const double2* amps, u64 n, u32 M, u64* smp, cudaStream_t st, const u64* keys = nullptr, const PendPred* pd = nullptr,
                  const GateTab* xf_tab = nullptr);
int svk_ss_pivot(const u64* smp_sorted, u32 M, u64 n_live, u64 max_terms, double min_mass, double mass_est, SampleCtl* ctl,
                 cudaStream_t st, const PreCut* pre = nullptr);
int svk_ss_classify(const u64* keys, const double2* amps, u64 n, SampleCtl* ctl, u64* ckeys, double2* camps, unsigned char* seg_cnt,
                    cudaStream_t st, double2* amps_rw = nullptr, const PendPred* pd = nullptr, const GateTab* xf_tab = nullptr);
// squeeze out the entries below the sampled band (uses the classify pass's per-segment counts)
int svk_ss_band_compact(const u64* keys, const double2* amps, u64 n, const SampleCtl* ctl, const unsigned char* seg_cnt,
                        u32* chunk_cnt, u64* scan_status, u32* tile_counter, u64* kout, double2* aout, cudaStream_t st);
int svk_scan_u32(u32* data, u64 n, u64* status, u32* tile_counter, cudaStream_t st);
int svk_sel_seed(SelState* ss, u64* hist, const SampleCtl* ctl, u64 n_orig, u64 max_terms, double min_mass, cudaStream_t st,
                 const PreCut* pre = nullptr);
int svk_compact(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n,
                const PendPred& pd, u64* status, u32* tile_counter, u64* d_count, cudaStream_t st);

int svk_check(const u64* keys, const double2* amps, u64 n, int nq, int* d_bad, cudaStream_t st);

// readout / load helpers
int svk_gather_top(const u64* keys, const double2* amps, u64 n, const SelState* ss, int use_sel,
                   KeyMap km, u64* o_pat, u64* o_lkey, double2* o_amp, u64* d_count, u64 kmax,
                   cudaStream_t st);
int svk_sort_pairs(u64* keys, u32* vals, u64* keys_alt, u32* vals_alt, u64 n, int bits,
                   u32* hist_scratch, cudaStream_t st, int* result_in_alt);
size_t svk_sort_scratch_bytes(u64 n);
int svk_iota(u32* v, u64 n, cudaStream_t st);
int svk_gather_u64(const u64* src, const u32* idx, u64* dst, u64 n, int invert, cudaStream_t st);
int svk_gather_c128(const double2* src, const u32* idx, double2* dst, u64 n, cudaStream_t st);
int svk_pat_to_prob(const u64* pat, double* prob, u64 n, cudaStream_t st);

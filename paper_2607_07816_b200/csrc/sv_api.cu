// Host side of the C ABI (include/sparse_sv.h): state, gate classification (SURVEY.md row
// a-1), pass planning, truncation driver, readout and load.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "../../include/sparse_sv.h"
#include "sv_internal.h"

struct sv_state {
    int n;
    u64 cap;
    cudaStream_t stream;
    bool own_mem, own_stream;
    unsigned char* arena;
    u64* keys[2];
    double2* amps[2];
    int cur;
    u64 count;   // logical number of terms
    u64 phys;    // stored entries in the current buffers (> count while a truncation is deferred)
    PendPred defer;   // truncation whose compaction is left to the next reader of the state
    // physical layout: stored bit phys_of_log[q] holds logical qubit q (XOR the lazy X mask)
    int phys_of_log[64];
    u64 xmask;   // in physical positions
    // device scratch
    TileDesc* desc;
    u64* status;
    u64* hist;
    SelState* sel;
    GateTab* tab;
    u64* d_count;
    u32* tile_counter;
    int* d_bad;
    double* partials;
    double* d_norm;
    u64* lut;          // device, 8 x 256: stored -> logical key tables of the current layout
    bool lut_valid;
    unsigned char* pinned;   // host, for small read-backs
    sv_stats stats;
    char err[256];
    // optional per-kernel timing (sv_profile): CUDA events around the main kernels
    bool prof_on;
    int npend;
    struct { int id; double bytes; } pend[64];
    cudaEvent_t evpool[128];
    bool ev_ready;
    sv_kernel_prof prof[SV_K_COUNT];
    // sampled fast path of the truncation cut
    SampleCtl* sctl;
    u64* smp_k[2];
    u32* smp_v[2];
    u32* smp_scr;
    unsigned char* seg_cnt;  // per 32-entry segment: entries not below the sampled band (band compaction)
    u32* chunk_cnt;          // per 1024-entry chunk: their sum, then the exclusive scan
    bool band_valid;         // the last select ran through the sampled path: seg_cnt / sctl describe the current arrays
    u64 band_above, band_cand;
    u64 sample_min_terms;   // states with fewer terms use the full-state select
    double mass_est;        // total mass of the current state if known (NaN: unknown); gates are taken as unitary
    // fused apply + truncate (sv_presample.cu)
    PreCut* pre;            // device: floor of the running gate, then count / mass of the outputs it left out
    u64 fuse_K;             // != 0 while sv_apply_gate runs on behalf of sv_apply_gate_truncate: the cap that follows
    bool pre_valid;         // the current arrays lack pre_cnt outputs of the last gate (all below every stored term)
    u64 pre_cnt;
    bool fuse_on;           // sv_apply_gate runs on behalf of sv_apply_gate_truncate
    bool diag_deferred;     // the diagonal gate in s->tab (and the pending cut) has not been applied yet: the truncation's
                            // classification pass applies it in place (sv_sample_select.cu, XF)
    bool small_on;          // SV_OPT_SMALL_STATE_PATH: sv_apply_circuit may use the single-block path (sv_small.cu)
    int two_bit_min_ma;     // SV_OPT_TWO_BIT_PASS: the final pass of a dense gate with at least this many active qubits moves two bits at once (0: never)
    u64 small_gates;        // gates it has taken so far
    int circuit_done;       // gates the running / last sv_apply_circuit completed
    int small_backoff;      // gates still to take the streaming passes after a gate that did not fit the small path ...
    u64 small_fail_work;    // ... unless their bound count * 2^m is below this one (that of the gate that failed)
    long long pre_slack;    // sv_test_set_pre_slack: sample points added to the floor's margin (tests force a failed margin with < 0)
};
#define SV_SAMPLE_MAX (1u << 16)

static void prof_drain(sv_state* s) {
    if (!s->npend) return;
    cudaStreamSynchronize(s->stream);
    for (int i = 0; i < s->npend; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, s->evpool[2 * i], s->evpool[2 * i + 1]) == cudaSuccess) {
            sv_kernel_prof& k = s->prof[s->pend[i].id];
            k.ms += ms; k.launches += 1; k.alg_bytes += s->pend[i].bytes;
        }
    }
    s->npend = 0;
}
// Reserve an event pair for one launch of kernel `id` moving `bytes` algorithmic bytes.
static void prof_slot(sv_state* s, int id, double bytes, cudaEvent_t* e0, cudaEvent_t* e1) {
    *e0 = *e1 = nullptr;
    if (!s->prof_on) return;
    if (s->npend == 64) prof_drain(s);
    s->pend[s->npend].id = id; s->pend[s->npend].bytes = bytes;
    *e0 = s->evpool[2 * s->npend]; *e1 = s->evpool[2 * s->npend + 1];
    s->npend += 1;
}

int sv_cur_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) dev = 0;
    return dev < SV_MAX_DEV ? dev : SV_MAX_DEV - 1;
}
int sv_sm_count() {   // per device; concurrent first calls write the same value
    static int n[SV_MAX_DEV];
    const int dev = sv_cur_device();
    if (!n[dev]) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v < 1) v = 148;
        n[dev] = v;
    }
    return n[dev];
}

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }
static u64 desc_entries(u64 cap) { return cap / 112 + 8; }

struct ArenaLayout { size_t keys[2], amps[2], desc, status, hist, sel, tab, misc, partials, lut, sctl, pre, smp_k[2], smp_v[2], smp_scr, seg_cnt, chunk_cnt, total; };
static ArenaLayout layout_for(u64 cap) {
    ArenaLayout L; size_t o = 0;
    for (int i = 0; i < 2; ++i) { L.keys[i] = o; o += align_up(cap * 8); }
    for (int i = 0; i < 2; ++i) { L.amps[i] = o; o += align_up(cap * 16); }
    L.desc = o; o += align_up(desc_entries(cap) * sizeof(TileDesc));
    L.status = o; o += align_up(desc_entries(cap) * 8);
    L.hist = o; o += align_up(3 * SV_SEL_BINS * 8);   // >= the select's 5 x 2048 + 8 words
    L.sel = o; o += align_up(sizeof(SelState));
    L.tab = o; o += align_up(sizeof(GateTab));
    L.misc = o; o += 256;
    L.partials = o; o += align_up(1024 * 8 + 8);
    L.lut = o; o += align_up(8 * 256 * 8);
    L.sctl = o; o += align_up(sizeof(SampleCtl));
    L.pre = o; o += align_up(sizeof(PreCut));
    for (int i = 0; i < 2; ++i) { L.smp_k[i] = o; o += align_up((size_t)SV_SAMPLE_MAX * 8); }
    for (int i = 0; i < 2; ++i) { L.smp_v[i] = o; o += align_up((size_t)SV_SAMPLE_MAX * 4); }
    L.smp_scr = o; o += align_up(svk_sort_scratch_bytes(SV_SAMPLE_MAX));
    L.seg_cnt = o; o += align_up(cap / 32 + 256);
    L.chunk_cnt = o; o += align_up((cap / 1024 + 8) * 4);
    L.total = o;
    return L;
}

static int fail(sv_state* s, int code, const char* msg) {
    if (s) snprintf(s->err, sizeof(s->err), "%s", msg);
    return code;
}
static int cuda_fail(sv_state* s, cudaError_t e, const char* where) {
    if (s) snprintf(s->err, sizeof(s->err), "%s: %s", where, cudaGetErrorString(e));
    return SV_ERR_CUDA;
}
#define CU(call)                                                           \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) return cuda_fail(s, e__, #call);           \
    } while (0)
// Debug builds only (-DSV_DEBUG_SYNC): synchronise after every kernel of the truncation path and name the first
// one that failed.  The release library has no such code path.
#ifdef SV_DEBUG_SYNC
#define DBG_SYNC(tag)                                                                            \
    do {                                                                                         \
        cudaError_t e__ = cudaStreamSynchronize(s->stream);                                      \
        if (e__ != cudaSuccess) return cuda_fail(s, e__, tag);                                   \
    } while (0)
#else
#define DBG_SYNC(tag) do { } while (0)
#endif
#define CHECK_LAUNCH()                                                     \
    do {                                                                   \
        cudaError_t e__ = cudaGetLastError();                              \
        if (e__ != cudaSuccess) return cuda_fail(s, e__, "kernel launch"); \
    } while (0)

// Builds (if the layout changed) and uploads the stored -> logical key tables.
static KeyMap keymap_of(sv_state* s) {
    if (!s->lut_valid) {
        static thread_local u64 h[8 * 256];
        u64 col[64];
        for (int p = 0; p < 64; ++p) col[p] = 0;
        for (int q = 0; q < s->n; ++q) col[s->phys_of_log[q]] = 1ull << q;
        u64 xl = 0;
        for (int p = 0; p < 64; ++p) if ((s->xmask >> p) & 1ull) xl ^= col[p];
        for (int b = 0; b < 8; ++b)
            for (int v = 0; v < 256; ++v) {
                u64 o = (b == 0) ? xl : 0;
                for (int j = 0; j < 8; ++j) if ((v >> j) & 1) o ^= col[8 * b + j];
                h[b * 256 + v] = o;
            }
        cudaMemcpyAsync(s->lut, h, sizeof(h), cudaMemcpyHostToDevice, s->stream);
        s->lut_valid = true;
    }
    KeyMap km; km.lut = s->lut;
    return km;
}

// move physical bit p to position 0 (bits below p shift up by one)
static void layout_move(sv_state* s, int p) {
    s->lut_valid = false;
    for (int q = 0; q < s->n; ++q) {
        if (s->phys_of_log[q] < p) s->phys_of_log[q] += 1;
        else if (s->phys_of_log[q] == p) s->phys_of_log[q] = 0;
    }
    const u64 low = (p == 0) ? 0 : (s->xmask & ((1ull << p) - 1));
    const u64 hi = (p == 63) ? 0 : (s->xmask & ~((2ull << p) - 1));
    s->xmask = hi | (low << 1) | ((s->xmask >> p) & 1ull);
}

extern "C" size_t sv_arena_bytes(uint64_t capacity) { return layout_for(capacity).total; }

static int init_state(sv_state* s) {
    s->cur = 0;
    s->count = 1; s->phys = 1;
    s->defer.active = 0;
    s->lut_valid = false;
    s->mass_est = 1.0;
    s->xmask = 0;
    for (int q = 0; q < 64; ++q) s->phys_of_log[q] = q;
    const u64 k0 = 0;
    const double2 a0 = make_double2(1.0, 0.0);   // ground state
    CU(cudaMemcpyAsync(s->keys[0], &k0, 8, cudaMemcpyHostToDevice, s->stream));
    CU(cudaMemcpyAsync(s->amps[0], &a0, 16, cudaMemcpyHostToDevice, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    return SV_OK;
}

static int create_common(int n_qubits, uint64_t capacity, void* arena, size_t arena_bytes, void* stream, bool own,
                         sv_state** out) {
    if (!out) return SV_ERR_INVALID_ARG;
    *out = nullptr;
    if (n_qubits < 1 || n_qubits > 64 || capacity < 1 || capacity >= (1ull << 32) * 8) return SV_ERR_INVALID_ARG;
    const ArenaLayout L = layout_for(capacity);
    sv_state* s = new (std::nothrow) sv_state();
    if (!s) return SV_ERR_NOMEM;
    memset(s, 0, sizeof(*s));
    s->n = n_qubits; s->cap = capacity; s->own_mem = own; s->own_stream = own;
    if (own) {
        if (cudaMalloc(&arena, L.total) != cudaSuccess) { cudaGetLastError(); delete s; return SV_ERR_NOMEM; }
        cudaStream_t st;
        if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) { cudaFree(arena); delete s; return SV_ERR_CUDA; }
        s->stream = st;
    } else {
        if (!arena || arena_bytes < L.total || ((uintptr_t)arena & 255)) { delete s; return SV_ERR_INVALID_ARG; }
        s->stream = (cudaStream_t)stream;
    }
    s->arena = (unsigned char*)arena;
    for (int i = 0; i < 2; ++i) { s->keys[i] = (u64*)(s->arena + L.keys[i]); s->amps[i] = (double2*)(s->arena + L.amps[i]); }
    s->desc = (TileDesc*)(s->arena + L.desc);
    s->status = (u64*)(s->arena + L.status);
    s->hist = (u64*)(s->arena + L.hist);
    s->sel = (SelState*)(s->arena + L.sel);
    s->tab = (GateTab*)(s->arena + L.tab);
    s->d_count = (u64*)(s->arena + L.misc);
    s->tile_counter = (u32*)(s->arena + L.misc + 64);
    s->d_bad = (int*)(s->arena + L.misc + 128);
    s->d_norm = (double*)(s->arena + L.misc + 192);
    s->partials = (double*)(s->arena + L.partials);
    s->lut = (u64*)(s->arena + L.lut);
    s->sctl = (SampleCtl*)(s->arena + L.sctl);
    s->pre = (PreCut*)(s->arena + L.pre);
    for (int i = 0; i < 2; ++i) { s->smp_k[i] = (u64*)(s->arena + L.smp_k[i]); s->smp_v[i] = (u32*)(s->arena + L.smp_v[i]); }
    s->smp_scr = (u32*)(s->arena + L.smp_scr);
    s->seg_cnt = s->arena + L.seg_cnt;
    s->chunk_cnt = (u32*)(s->arena + L.chunk_cnt);
    s->small_on = true;
    s->two_bit_min_ma = 3;
    s->sample_min_terms = 1ull << 21;   // below ~2^21 terms the state sits in L2 and the full select has fewer launches
    if (cudaMallocHost(&s->pinned, 1024) != cudaSuccess) { if (own) { cudaFree(arena); cudaStreamDestroy(s->stream); } delete s; return SV_ERR_NOMEM; }
    if (cudaMemsetAsync(s->hist, 0, 3 * SV_SEL_BINS * 8, s->stream) != cudaSuccess || init_state(s) != SV_OK) {
        sv_destroy(s);
        return SV_ERR_CUDA;
    }
    *out = s;
    return SV_OK;
}

extern "C" int sv_create(int n_qubits, uint64_t capacity, sv_state** out) {
    return create_common(n_qubits, capacity, nullptr, 0, nullptr, true, out);
}
extern "C" int sv_create_in_arena(int n_qubits, uint64_t capacity, void* dev_arena, size_t arena_bytes, void* cuda_stream,
                                  sv_state** out) {
    return create_common(n_qubits, capacity, dev_arena, arena_bytes, cuda_stream, false, out);
}
extern "C" void sv_destroy(sv_state* s) {
    if (!s) return;
    cudaStreamSynchronize(s->stream);
    if (s->ev_ready) for (int i = 0; i < 128; ++i) cudaEventDestroy(s->evpool[i]);
    if (s->pinned) cudaFreeHost(s->pinned);
    if (s->own_mem && s->arena) cudaFree(s->arena);
    if (s->own_stream && s->stream) cudaStreamDestroy(s->stream);
    delete s;
}
extern "C" const char* sv_last_error(const sv_state* s) { return s ? s->err : "null handle"; }
extern "C" int sv_sync(sv_state* s) {
    if (!s) return SV_ERR_INVALID_ARG;
    CU(cudaStreamSynchronize(s->stream));
    return SV_OK;
}
extern "C" int sv_num_terms(sv_state* s, uint64_t* n) {
    if (!s || !n) return SV_ERR_INVALID_ARG;
    CU(cudaStreamSynchronize(s->stream));
    *n = s->count;
    return SV_OK;
}
extern "C" int sv_profile(sv_state* s, int enable) {
    if (!s) return SV_ERR_INVALID_ARG;
    prof_drain(s);
    if (enable && !s->ev_ready) {
        for (int i = 0; i < 128; ++i) CU(cudaEventCreate(&s->evpool[i]));
        s->ev_ready = true;
    }
    memset(s->prof, 0, sizeof(s->prof));
    s->prof_on = enable != 0;
    return SV_OK;
}
extern "C" int sv_profile_get(sv_state* s, int kernel, sv_kernel_prof* out) {
    if (!s || !out || kernel < 0 || kernel >= SV_K_COUNT) return SV_ERR_INVALID_ARG;
    prof_drain(s);
    *out = s->prof[kernel];
    return SV_OK;
}
extern "C" int sv_set_option(sv_state* s, int option, uint64_t value) {
    if (!s) return SV_ERR_INVALID_ARG;
    if (option == SV_OPT_SAMPLE_MIN_TERMS) { s->sample_min_terms = value; return SV_OK; }
    if (option == SV_OPT_SMALL_STATE_PATH) { s->small_on = value != 0; return SV_OK; }
    if (option == SV_OPT_TWO_BIT_PASS) { s->two_bit_min_ma = value == 0 ? 0 : (value == 1 ? 2 : 3); return SV_OK; }
    return fail(s, SV_ERR_INVALID_ARG, "unknown option");
}
// test hook (include/sparse_sv_test.h): sample points added to the margin of the fused call's output floor
extern "C" int sv_test_set_pre_slack(sv_state* s, long long slack) {
    if (!s) return SV_ERR_INVALID_ARG;
    s->pre_slack = slack;
    return SV_OK;
}
// test / diagnostic hook (include/sparse_sv_test.h): bit q of *mask is set iff qubit q has the same value in every term
extern "C" int sv_test_definite_qubits(sv_state* s, uint64_t* mask) {
    if (!s || !mask) return SV_ERR_INVALID_ARG;
    svk_key_masks(s->keys[s->cur], s->amps[s->cur], s->phys, s->defer, 1, s->d_count + 4, s->stream);
    u64 oa[2] = {0, 0};
    CU(cudaMemcpyAsync(s->pinned, s->d_count + 4, sizeof(oa), cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    memcpy(oa, s->pinned, sizeof(oa));
    const u64 same = ~(oa[0] ^ oa[1]);
    u64 m = 0;
    for (int q = 0; q < s->n; ++q) if ((same >> s->phys_of_log[q]) & 1ull) m |= 1ull << q;
    *mask = (s->count == 0) ? 0 : m;
    return SV_OK;
}
extern "C" int sv_get_stats(sv_state* s, sv_stats* out) {
    if (!s || !out) return SV_ERR_INVALID_ARG;
    s->stats.small_gates = s->small_gates;
    *out = s->stats;
    return SV_OK;
}

static int read_back(sv_state* s, void* dst, const void* dsrc, size_t bytes) {
    CU(cudaMemcpyAsync(s->pinned, dsrc, bytes, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    memcpy(dst, s->pinned, bytes);
    return SV_OK;
}

// Apply a deferred truncation and squeeze out dead entries now (one compaction pass).  Readers that
// cannot fuse the predicate into their own load, or that need a dense array, call this first.
static int materialize(sv_state* s) {
    if (!s->defer.active && s->phys == s->count) return SV_OK;
    const int alt = s->cur ^ 1;
    cudaEvent_t e0, e1;
    prof_slot(s, SV_K_COMPACT, 24.0 * ((double)s->phys + (double)s->count), &e0, &e1);
    if (e0) cudaEventRecord(e0, s->stream);
    s->stats.launches += svk_compact(s->keys[s->cur], s->amps[s->cur], s->keys[alt], s->amps[alt], s->phys, s->defer,
                                     s->status, s->tile_counter, s->d_count, s->stream);
    if (e1) cudaEventRecord(e1, s->stream);
    CHECK_LAUNCH();
    s->stats.passes += 1;
    s->cur = alt;
    s->phys = s->count;
    s->defer.active = 0;
    return SV_OK;
}
// Dead entries (terms dropped in place) are tolerated up to 1/8 of the live terms.
static inline bool few_dead(const sv_state* s) { return s->phys - s->count <= s->count / 8; }

// In-place diagonal gate from s->tab, fused with a pending truncation if there is one (few dead entries).
static int launch_diag_in_place(sv_state* s) {
    cudaEvent_t e0, e1;
    prof_slot(s, SV_K_DIAG, 40.0 * (double)s->phys, &e0, &e1);
    if (e0) cudaEventRecord(e0, s->stream);
    if (s->defer.active) {   // dropped terms become dead entries
        s->stats.launches += svk_diag_pend(s->keys[s->cur], s->amps[s->cur], s->phys, s->tab, 1, s->defer, s->stream);
        s->defer.active = 0;
    } else {
        s->stats.launches += svk_diag(s->keys[s->cur], s->amps[s->cur], s->phys, s->tab, s->stream);
    }
    if (e1) cudaEventRecord(e1, s->stream);
    CHECK_LAUNCH();
    return SV_OK;
}
static int flush_diag(sv_state* s) {
    if (!s->diag_deferred) return SV_OK;
    s->diag_deferred = false;
    return launch_diag_in_place(s);
}

// ---------------------------------------------------------------------------------------
// sv_apply_gate: classify (row a-1), plan the bit moves, launch
// ---------------------------------------------------------------------------------------
static inline bool is_zero(const sv_c128& z) { return z.re == 0.0 && z.im == 0.0; }

extern "C" int sv_apply_gate(sv_state* s, const int* qubits, int m, const sv_c128* U) {
    if (!s || !qubits || !U) return s ? fail(s, SV_ERR_INVALID_ARG, "null argument") : SV_ERR_INVALID_ARG;
    if (m < 1 || m > SV_MAX_M) return fail(s, SV_ERR_INVALID_ARG, "m must be 1..4");
    u64 seen = 0;
    for (int j = 0; j < m; ++j) {
        if (qubits[j] < 0 || qubits[j] >= s->n) return fail(s, SV_ERR_INVALID_ARG, "qubit out of range");
        if (seen & (1ull << qubits[j])) return fail(s, SV_ERR_INVALID_ARG, "repeated qubit");
        seen |= 1ull << qubits[j];
    }
    const int d = 1 << m;
    s->err[0] = 0;
    s->pre_valid = false;
    s->stats.pre_dropped = 0; s->stats.n_mid = 0;
    s->stats.m = m; s->stats.n_in = s->count; s->stats.n_out = s->count; s->stats.passes = 0;

    // a-1: bit j is control-like iff U never connects patterns that differ in bit j
    int active[SV_MAX_M], ctrl[SV_MAX_M], ma = 0, mc = 0;
    for (int j = 0; j < m; ++j) {
        bool mixes = false;
        for (int r = 0; r < d && !mixes; ++r)
            for (int c = 0; c < d; ++c)
                if ((((r ^ c) >> j) & 1) && !is_zero(U[r * d + c])) { mixes = true; break; }
        if (mixes) active[ma++] = j; else ctrl[mc++] = j;
    }
    s->stats.active_bits = ma;
    int amask_l = 0;
    for (int i = 0; i < ma; ++i) amask_l |= 1 << active[i];
    // lazy X mask on the gate's qubits, as a local pattern
    int xm = 0;
    for (int j = 0; j < m; ++j) xm |= (int)((s->xmask >> s->phys_of_log[qubits[j]]) & 1ull) << j;
    auto Ueff = [&](int r, int c) -> const sv_c128& { return U[(r ^ xm) * d + (c ^ xm)]; };   // in stored patterns

    GateTab tab;
    memset(&tab, 0, sizeof(tab));
    if (s->count == 0) { s->stats.gate_class = SV_CLASS_NONE; return SV_OK; }

    // Relabelling class (rows a-3, f-4): U is monomial and its nonzero of column c sits in row sigma(c) = pi(c) ^ x0 with
    // pi a PERMUTATION OF THE GATE'S QUBITS and x0 a constant pattern -- X, SWAP, any product of them, with phases.  Such a
    // gate only renames qubits and flips bits: the lazy layout (phys_of_log, xmask) takes it, no data is touched
    // ("just permutes the amplitudes"); phases, if any, go through the diagonal pass.
    bool xor_class = ma > 0, diag_nonzero = true, unit_phase = true;
    int sigma[16], pi[SV_MAX_M] = {0, 1, 2, 3}, x0 = 0;
    for (int c = 0; c < d && xor_class; ++c) {
        int nz = 0;
        for (int r = 0; r < d; ++r) if (!is_zero(U[r * d + c])) { sigma[c] = r; ++nz; }
        if (nz != 1) xor_class = false;
    }
    if (xor_class) {
        x0 = sigma[0];
        int used = 0;
        for (int j = 0; j < m && xor_class; ++j) {
            const int v = sigma[1 << j] ^ x0;
            if (v == 0 || (v & (v - 1)) || (used & v)) { xor_class = false; break; }
            used |= v;
            pi[j] = __builtin_ctz((unsigned)v);
        }
        for (int c = 0; c < d && xor_class; ++c) {
            int pc = 0;
            for (int j = 0; j < m; ++j) pc |= ((c >> j) & 1) << pi[j];
            if (sigma[c] != (pc ^ x0)) xor_class = false;
        }
    }
    if (ma == 0)
        for (int c = 0; c < d; ++c) if (is_zero(U[c * d + c])) diag_nonzero = false;

    // (ma == 0 with an exact zero on the diagonal -- a projector: U is not required to be unitary -- is still a diagonal
    // gate; the terms it annihilates are dropped: they become dead entries and are counted below.)
    if (ma == 0 || xor_class) {
        // phase table in stored patterns: every gate bit acts as a control of a diagonal
        tab.ma = 0; tab.mc = m;
        for (int j = 0; j < m; ++j) tab.ctrl_pos[j] = s->phys_of_log[qubits[j]];
        for (int cs = 0; cs < d; ++cs) {
            const int ct = cs ^ xm;                       // true pattern of the stored pattern
            const sv_c128 z = U[(xor_class ? sigma[ct] : ct) * d + ct];
            tab.U[cs] = make_double2(z.re, z.im);
            if (!(z.re == 1.0 && z.im == 0.0)) unit_phase = false;
        }
        if (xor_class) {   // new layout: qubit qubits[pi[j]] now lives where qubits[j] lived, flipped if x0 says so -- no data is touched
            int oldp[SV_MAX_M];
            for (int j = 0; j < m; ++j) oldp[j] = s->phys_of_log[qubits[j]];
            for (int j = 0; j < m; ++j) {
                s->phys_of_log[qubits[pi[j]]] = oldp[j];
                if ((x0 >> pi[j]) & 1) s->xmask ^= 1ull << oldp[j];
            }
            s->lut_valid = false;
        }
        s->stats.gate_class = xor_class ? SV_CLASS_XOR : SV_CLASS_DIAGONAL;
        if (!unit_phase) {
            CU(cudaMemcpyAsync(s->tab, &tab, sizeof(tab), cudaMemcpyHostToDevice, s->stream));
            cudaEvent_t e0, e1;
            if (s->defer.active && !few_dead(s)) {   // truncate-then-diagonal in one out-of-place, compacting pass
                const int alt = s->cur ^ 1;
                prof_slot(s, SV_K_DIAG, 24.0 * ((double)s->phys + (double)s->count), &e0, &e1);
                if (e0) cudaEventRecord(e0, s->stream);
                s->stats.launches += svk_diag_compact(s->keys[s->cur], s->amps[s->cur], s->keys[alt], s->amps[alt], s->phys,
                                                      s->tab, s->defer, s->status, s->tile_counter, s->d_count, s->stream);
                if (e1) cudaEventRecord(e1, s->stream);
                s->cur = alt; s->phys = s->count; s->defer.active = 0;
            } else if (diag_nonzero && s->fuse_on && s->count >= s->sample_min_terms && s->phys / 8 >= 64) {
                // fused call: the sampled truncation that follows applies the gate in its own pass over the state
                s->diag_deferred = true;
            } else {
                int rcd = launch_diag_in_place(s);
                if (rcd != SV_OK) return rcd;
            }
            CHECK_LAUNCH();
            s->stats.passes = 1;
            if (!diag_nonzero) {   // singular diagonal: count what is left
                s->stats.launches += svk_count_live(s->amps[s->cur], s->phys, s->d_count, s->stream);
                CHECK_LAUNCH();
                u64 live = 0;
                int rcl = read_back(s, &live, s->d_count, sizeof(u64));
                if (rcl != SV_OK) return rcl;
                s->count = live;
                if (live == 0) s->phys = 0;
                s->mass_est = nan("");
                s->stats.n_out = live;
            }
        }
        return SV_OK;
    }
    if (ma < 1) return fail(s, SV_ERR_INVALID_ARG, "internal: gate without an active qubit in the group class");

    // GROUP class.  The active bits must occupy physical positions 0..ma-1.  Those already
    // forming a prefix {0..k-1} stay; the others are moved to the LSB one pass each, the
    // last move fused with the tuple mat-vec.
    s->stats.gate_class = SV_CLASS_GROUP;
    int need[SV_MAX_M], nneed = 0;
    {
        bool inlow[SV_MAX_M + 1] = {false, false, false, false, false};
        for (int i = 0; i < ma; ++i) { const int p = s->phys_of_log[qubits[active[i]]]; if (p < ma) inlow[p] = true; }
        int k = 0;
        while (k < ma && inlow[k]) ++k;
        for (int i = ma - 1; i >= 0; --i)
            if (s->phys_of_log[qubits[active[i]]] >= k) need[nneed++] = active[i];
    }
    // A dense gate (every entry of U nonzero: Haar SU(4), 8x8, 16x16) brings its LAST TWO missing bits down in the final pass
    // itself (a four-way merge per tile, sv_dense.cu TWO): one full pass over the state less.
    bool dense0 = (ma >= 2 && mc == 0);
    for (int i = 0; i < d * d && dense0; ++i) dense0 = !is_zero(U[i]);
    // (never inside the fused call: the fused variant of the two-bit pass, 2 resident blocks per SM, measured 1 to 5 % slower than
    // move + final pass -- profiles/r2_final.md -- and is not built)
    const bool two = s->two_bit_min_ma != 0 && ma >= s->two_bit_min_ma && dense0 && nneed >= 2 && s->fuse_K == 0;
    for (int t = 0; t + (two ? 2 : 1) < nneed; ++t) {   // pure moves: state preserving, committed one by one
        const int p = s->phys_of_log[qubits[need[t]]];
        if (p == 0) continue;
        const int alt = s->cur ^ 1;
        const int fixed = few_dead(s) ? 1 : 0;   // position preserving (dead entries carried) or compacting
        cudaEvent_t e0, e1;
        prof_slot(s, SV_K_MOVE, 24.0 * ((double)s->phys + (double)(fixed ? s->phys : s->count)), &e0, &e1);
        s->stats.launches += svk_bitpass(s->keys[s->cur], s->amps[s->cur], s->keys[alt], s->amps[alt], s->phys, p, 0, fixed, nullptr,
                                         s->defer, s->desc, s->status, s->tile_counter, s->d_count, s->cap, s->stream, e0, e1);
        CHECK_LAUNCH();
        s->cur = alt;
        if (!fixed) s->phys = s->count;      // dropped terms and dead entries have been squeezed out
        s->defer.active = 0;                 // a deferred truncation has been applied by the pass
        layout_move(s, p);
        s->stats.passes += 1;
    }
    int plast = -1, plast2 = -1;   // the bit(s) the final pass moves; two: plast > plast2
    if (nneed > 0) {
        plast = s->phys_of_log[qubits[need[nneed - 1]]];
        if (plast == 0) plast = -1;
    }
    if (two) {
        const int pa = s->phys_of_log[qubits[need[nneed - 2]]], pb = s->phys_of_log[qubits[need[nneed - 1]]];
        plast = pa > pb ? pa : pb; plast2 = pa > pb ? pb : pa;
    }
    // layout after the final move (on a copy: committed only on success)
    sv_state after = *s;
    if (plast > 0) layout_move(&after, plast);
    if (two) layout_move(&after, plast2 + 1);   // (the lower bit has moved up by one)
    tab.ma = ma; tab.mc = mc;
    int fpos[SV_MAX_M];
    for (int i = 0; i < ma; ++i) fpos[i] = after.phys_of_log[qubits[active[i]]];   // in 0..ma-1
    for (int i = 0; i < mc; ++i) tab.ctrl_pos[i] = after.phys_of_log[qubits[ctrl[i]]];
    for (int t = 0; t < (1 << ma); ++t) {
        int x = 0;
        for (int i = 0; i < ma; ++i) x |= ((t >> i) & 1) << fpos[i];
        tab.colorder[t] = x;
    }
    for (int cx = 0; cx < (1 << mc); ++cx)
        for (int xr = 0; xr < (1 << ma); ++xr)
            for (int xc = 0; xc < (1 << ma); ++xc) {
                int r = 0, c = 0;
                for (int i = 0; i < mc; ++i) { r |= ((cx >> i) & 1) << ctrl[i]; c |= ((cx >> i) & 1) << ctrl[i]; }
                for (int i = 0; i < ma; ++i) { r |= ((xr >> fpos[i]) & 1) << active[i]; c |= ((xc >> fpos[i]) & 1) << active[i]; }
                const sv_c128& z = Ueff(r, c);
                tab.U[(((cx << ma) | xr) << ma) | xc] = make_double2(z.re, z.im);
            }
    CU(cudaMemcpyAsync(s->tab, &tab, sizeof(tab), cudaMemcpyHostToDevice, s->stream));
    const int alt = s->cur ^ 1;
    cudaEvent_t ge0, ge1;
    // one active bit whose 2x2 blocks are all monomial (CNOT, Toffoli, ...): every stored entry maps to
    // exactly one stored entry, the pass needs no scan and the term count is known without a read-back
    bool monomial = (ma == 1);
    for (int cx = 0; cx < (1 << mc) && monomial; ++cx) {
        const double2* u = &tab.U[cx << 2];
        const bool z00 = u[0].x == 0.0 && u[0].y == 0.0, z01 = u[1].x == 0.0 && u[1].y == 0.0;
        const bool z10 = u[2].x == 0.0 && u[2].y == 0.0, z11 = u[3].x == 0.0 && u[3].y == 0.0;
        monomial = (!z00 && !z11 && z01 && z10) || (z00 && z11 && !z01 && !z10);
    }
    if (ma == 1 && monomial && plast < 0) {
        // the active bit already is the physical LSB: partners are stored neighbours, the gate is applied IN PLACE (row f-4)
        prof_slot(s, SV_K_DIAG, 40.0 * (double)s->phys, &ge0, &ge1);
        if (ge0) cudaEventRecord(ge0, s->stream);
        s->stats.launches += svk_perm_lsb(s->keys[s->cur], s->amps[s->cur], s->phys, s->tab, s->defer, s->stream);
        if (ge1) cudaEventRecord(ge1, s->stream);
        CHECK_LAUNCH();
        s->stats.passes += 1;
        s->defer.active = 0;
        s->stats.n_out = s->count;
        return SV_OK;
    }
    if (ma == 1 && monomial && few_dead(s)) {
        prof_slot(s, SV_K_BITPASS, 48.0 * (double)s->phys, &ge0, &ge1);
        s->stats.launches += svk_bitpass(s->keys[s->cur], s->amps[s->cur], s->keys[alt], s->amps[alt], s->phys, plast > 0 ? plast : 0, 2, 1,
                                         s->tab, s->defer, s->desc, s->status, s->tile_counter, s->d_count, s->cap, s->stream, ge0, ge1);
        CHECK_LAUNCH();
        s->stats.passes += 1;
        if (plast > 0) { memcpy(s->phys_of_log, after.phys_of_log, sizeof(s->phys_of_log)); s->xmask = after.xmask; s->lut_valid = false; }
        s->cur ^= 1;
        s->defer.active = 0;
        s->stats.n_out = s->count;
        return SV_OK;
    }
    const u64 n_live_in = s->count;
    bool dense = (ma >= 2 && mc == 0);   // every entry nonzero: each tuple yields exactly 2^ma outputs (sv_dense.cu)
    for (int i = 0; i < (1 << (2 * ma)) && dense; ++i) dense = !(tab.U[i].x == 0.0 && tab.U[i].y == 0.0);
    // Fused apply + truncate: when the cap that follows will cut deep into the gate's output, a floor for that
    // cut is estimated from a sample of the outputs, and the pass leaves out what lies below it.
    u64 preM = s->phys / 8;
    if (preM > SV_SAMPLE_MAX) preM = SV_SAMPLE_MAX;
    bool use_pre = s->fuse_K != 0 && s->count >= s->sample_min_terms && s->phys < (1ull << 32) && preM >= 64 &&
                   ((u64)1 << ma) * s->count > s->fuse_K + s->fuse_K / 8;
    s->stats.pre_dropped = 0;
    u64 nout = 0, ndead = 0, npre = 0;
    for (;;) {
        u32 pre_parts = 0;
        if (use_pre) {
            const u32 M = (u32)preM;
            if (ma == 1)
                s->stats.launches += svk_pre_sample1(s->keys[s->cur], s->amps[s->cur], s->phys, plast > 0 ? plast : 0, s->tab, s->defer, M,
                                                     s->smp_k[0], s->stream);
            else
                s->stats.launches += svk_pre_sample_group(s->keys[s->cur], s->amps[s->cur], s->phys, plast, ma, s->tab, s->defer, M,
                                                          s->smp_k[0], s->stream, plast2);
            int in_alt = 0;
            s->stats.launches += svk_sort_pairs(s->smp_k[0], s->smp_v[0], s->smp_k[1], s->smp_v[1], M, 24, s->smp_scr, s->stream, &in_alt);
            s->stats.launches += svk_pre_pivot(s->smp_k[in_alt ? 1 : 0], M, s->phys, 1u << ma, s->fuse_K, s->pre_slack, s->pre, s->stream);
            DBG_SYNC("pre_sample+pivot");
        }
        prof_slot(s, ma == 1 ? SV_K_BITPASS_GEN : SV_K_GROUPPASS, 0.0, &ge0, &ge1);
        const int gslot = s->npend - 1;
        double* pmass = reinterpret_cast<double*>(s->hist);          // per-block partials (the select's histogram is idle)
        u64* pcnt = s->hist + SV_SEL_BINS;
        if (ma == 1) {   // one active bit: the single-bit pass (p = 0 when the bit already sits at the LSB)
            s->stats.launches += svk_bitpass(s->keys[s->cur], s->amps[s->cur], s->keys[alt], s->amps[alt], s->phys, plast > 0 ? plast : 0, 1, 0,
                                             s->tab, s->defer, s->desc, s->status, s->tile_counter, s->d_count, s->cap, s->stream, ge0, ge1,
                                             use_pre ? s->pre : nullptr, pmass, pcnt, &pre_parts);
        } else {
            s->stats.launches += svk_grouppass(s->keys[s->cur], s->amps[s->cur], s->keys[alt], s->amps[alt], s->phys, plast, ma,
                                               s->tab, s->defer, s->desc, s->status, s->d_count, s->cap, s->stream, ge0, ge1,
                                               use_pre ? s->pre : nullptr, pmass, pcnt, &pre_parts, dense ? 1 : 0,
                                               // few dead entries: they ride along as zero members (their products add +-0: the
                                                // nonzero outputs keep their bits) -- unless the dead-only tuples' zero outputs
                                                // could then push a full-size output over the capacity
                                               (few_dead(s) && (s->phys << ma) <= s->cap) ? 0 : 1, plast2);
        }
        if (use_pre) s->stats.launches += svk_pre_finish(pmass, pcnt, pre_parts, s->pre, s->d_count, s->stream);
        CHECK_LAUNCH();
        s->stats.passes += 1;
        u64 cnts[3] = {0, 0, 0};   // stored outputs, dead ones among them (exact cancellations of a multi-bit gate), left out
        int rc = read_back(s, cnts, s->d_count, use_pre ? 3 * sizeof(u64) : (ma == 1 ? sizeof(u64) : 2 * sizeof(u64)));
        if (rc != SV_OK) return rc;
        nout = cnts[0]; ndead = (ma == 1) ? 0 : cnts[1]; npre = use_pre ? cnts[2] : 0;
        if (ge0) s->pend[gslot].bytes = 24.0 * ((double)n_live_in + (double)(nout > s->cap ? s->cap : nout));
        if (use_pre && npre > 0 && nout <= s->fuse_K) {   // the floor was too high (its margin failed): once more without it
            s->stats.fallbacks += 1;
            use_pre = false;
            continue;
        }
        break;
    }
    if (nout > s->cap) {
        s->stats.n_out = nout;
        return fail(s, SV_ERR_CAPACITY, "gate output exceeds capacity (state unchanged)");
    }
    if (plast > 0) { memcpy(s->phys_of_log, after.phys_of_log, sizeof(s->phys_of_log)); s->xmask = after.xmask; s->lut_valid = false; }
    s->cur ^= 1;
    s->count = nout - ndead; s->phys = nout;
    s->defer.active = 0;
    s->pre_valid = npre > 0; s->pre_cnt = npre;
    s->stats.n_out = s->count + npre; s->stats.pre_dropped = npre;
    return SV_OK;
}

// apply the (fused) gate, then truncate.  One call, so that the engine may let the gate's pass
// leave out what the cut is certain to drop (sv_presample.cu); the result is that of the two calls.
extern "C" int sv_apply_gate_truncate(sv_state* s, const int* qubits, int m, const sv_c128* U, uint64_t max_terms, double min_mass,
                                      double* kept_fraction) {
    if (!s) return SV_ERR_INVALID_ARG;
    if (!(min_mass > 0.0)) return fail(s, SV_ERR_INVALID_ARG, "min_mass must be > 0");
    s->fuse_K = max_terms; s->fuse_on = true;
    int rc = sv_apply_gate(s, qubits, m, U);
    s->fuse_K = 0; s->fuse_on = false;
    if (rc != SV_OK) { s->pre_valid = false; s->diag_deferred = false; return rc; }
    const sv_stats g = s->stats;
    if (s->diag_deferred && !((max_terms != 0 && max_terms < s->count) || min_mass < 1.0)) {   // the truncation will not look at the state
        rc = flush_diag(s);
        if (rc != SV_OK) return rc;
    }
    rc = sv_truncate(s, max_terms, min_mass, kept_fraction);
    s->pre_valid = false;
    if (s->diag_deferred) { const int rcf = flush_diag(s); if (rc == SV_OK) rc = rcf; }
    // statistics of the pair: the gate's class and passes, terms before the gate and after the cut
    const uint64_t n_kept = s->stats.n_out;
    const int tp = s->stats.passes;
    const uint64_t launches = s->stats.launches, fallbacks = s->stats.fallbacks;
    s->stats = g;
    s->stats.passes += tp; s->stats.launches = launches; s->stats.fallbacks = fallbacks;
    s->stats.n_mid = g.n_out;
    if (rc == SV_OK) s->stats.n_out = n_kept;
    return rc;
}

// ---------------------------------------------------------------------------------------
// sv_apply_circuit: a sequence of (gate, truncate) steps with look-ahead (row f-2; small states: H5)
// ---------------------------------------------------------------------------------------
#define SV_SMALL_BATCH 64
static int apply_circuit_impl(sv_state* s, int n_gates, const int* gate_m, const int* gate_qubits, const sv_c128* gate_U,
                              uint64_t max_terms, double min_mass, double* kept_fractions) {
    // offsets + validation of the whole list up front: an invalid gate anywhere leaves the state untouched
    size_t qoff = 0, uoff = 0;
    for (int g = 0; g < n_gates; ++g) {
        const int m = gate_m[g];
        if (m < 1 || m > SV_MAX_M) return fail(s, SV_ERR_INVALID_ARG, "sv_apply_circuit: m must be 1..4");
        u64 seen = 0;
        for (int j = 0; j < m; ++j) {
            const int q = gate_qubits[qoff + j];
            if (q < 0 || q >= s->n || (seen & (1ull << q))) return fail(s, SV_ERR_INVALID_ARG, "sv_apply_circuit: qubit out of range or repeated");
            seen |= 1ull << q;
        }
        qoff += m; uoff += (size_t)1 << (2 * m);
    }
    SmallGate* d_gates = reinterpret_cast<SmallGate*>(s->smp_k[0]);           // the sampling scratch is idle here
    double* d_kept = reinterpret_cast<double*>(s->smp_k[1]);
    SmallCtl* d_ctl = reinterpret_cast<SmallCtl*>(reinterpret_cast<unsigned char*>(s->smp_k[1]) + 1024);
    static_assert(sizeof(SmallGate) * SV_SMALL_BATCH <= (size_t)SV_SAMPLE_MAX * 8, "gate batch does not fit the scratch");
    SmallGate* h_gates = new (std::nothrow) SmallGate[SV_SMALL_BATCH];
    if (!h_gates) return fail(s, SV_ERR_NOMEM, "sv_apply_circuit: host allocation failed");
    int rc = SV_OK, g = 0;
    qoff = 0; uoff = 0;
    while (g < n_gates && rc == SV_OK) {
        // (after a gate that did not fit, a gate is tried on the small path again only if its bound count * 2^m is below that
        // of the gate that failed, or 16 gates later: a wasted launch + round trip costs about a third of a streaming gate)
        if (s->small_on && s->count > 0 && s->count <= SV_SMALL_CAP &&
            (s->small_backoff == 0 || (s->count << gate_m[g]) < s->small_fail_work)) {
            // ---- small-state batch: one single-block launch per gate, the count stays on the device ----
            rc = materialize(s);
            if (rc != SV_OK) break;
            const int B = (n_gates - g < SV_SMALL_BATCH) ? n_gates - g : SV_SMALL_BATCH;
            size_t qo = qoff, uo = uoff;
            for (int b = 0; b < B; ++b) {
                const int m = gate_m[g + b], d = 1 << m;
                SmallGate& sg = h_gates[b];
                memset(&sg, 0, sizeof(int) * (2 + SV_MAX_M));
                sg.m = m;
                for (int j = 0; j < m; ++j) {
                    const int ph = s->phys_of_log[gate_qubits[qo + j]];
                    sg.pos[j] = ph;
                    sg.xm |= (int)((s->xmask >> ph) & 1ull) << j;
                }
                for (int i = 0; i < d * d; ++i) sg.U[i] = make_double2(gate_U[uo + i].re, gate_U[uo + i].im);
                qo += m; uo += (size_t)d * d;
            }
            SmallCtl hc;
            memset(&hc, 0, sizeof(hc));
            hc.count = s->count; hc.fail_gate = -1;
            cudaStream_t st = s->stream;
            const KeyMap km = keymap_of(s);
            if (cudaMemcpyAsync(d_gates, h_gates, sizeof(SmallGate) * B, cudaMemcpyHostToDevice, st) != cudaSuccess ||
                cudaMemcpyAsync(d_ctl, &hc, sizeof(hc), cudaMemcpyHostToDevice, st) != cudaSuccess) { rc = cuda_fail(s, cudaGetLastError(), "sv_apply_circuit: upload"); break; }
            // block size: enough threads for the largest gate output this batch can see (count now or after a cap cut,
            // times 2^m, two entries per thread in the sorts), no more: its ~100 barriers per gate get cheaper with fewer warps
            u64 nmax = s->count;
            if (max_terms != 0 && max_terms > nmax) nmax = max_terms;
            if (max_terms == 0) nmax = SV_SMALL_CAP;
            int mmax = 1;
            for (int b = 0; b < B; ++b) if (gate_m[g + b] > mmax) mmax = gate_m[g + b];
            u64 work = (nmax << mmax) / 2;
            if (work < nmax) work = nmax;
            if (work > 1024) work = 1024;
            s->stats.launches += svk_small_gates(s->keys[s->cur], s->amps[s->cur], d_ctl, d_gates, B, km, max_terms, min_mass, d_kept, s->cap,
                                                 (int)work, st);
            if (cudaGetLastError() != cudaSuccess) { rc = fail(s, SV_ERR_CUDA, "sv_apply_circuit: kernel launch"); break; }
            struct { SmallCtl c; double kept[SV_SMALL_BATCH]; } back;
            // (ctl and the kept fractions are 1 KB apart in one scratch array: two small copies, one synchronisation)
            if (cudaMemcpyAsync(&back.c, d_ctl, sizeof(SmallCtl), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaMemcpyAsync(back.kept, d_kept, sizeof(double) * B, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
                cudaStreamSynchronize(st) != cudaSuccess) { rc = cuda_fail(s, cudaGetLastError(), "sv_apply_circuit: read-back"); break; }
            const int done = back.c.done_gates;
            if (done > 0) {
                s->stats.n_in = s->count; s->stats.n_mid = back.c.n_pre; s->stats.n_out = back.c.count;
                s->stats.gate_class = SV_CLASS_GROUP; s->stats.m = gate_m[g + done - 1]; s->stats.passes = done; s->stats.pre_dropped = 0;
                s->count = back.c.count; s->phys = back.c.count;
                s->mass_est = nan("");
                s->small_gates += (u64)done;
            }
            if (kept_fractions) for (int b = 0; b < done; ++b) kept_fractions[g + b] = back.kept[b];
            for (int b = 0; b < done; ++b) { qoff += gate_m[g + b]; uoff += (size_t)1 << (2 * gate_m[g + b]); }
            g += done;
            if (back.c.status) { s->small_backoff = 16; s->small_fail_work = s->count << gate_m[g]; }
            else s->small_backoff = 0;
            if (g >= n_gates || !back.c.status) continue;
            // gate g (or its output) does not fit one block: the streaming passes take it (and the loop comes back here
            // if the cut brings the state down again)
        }
        double kf = 1.0;
        rc = sv_apply_gate_truncate(s, gate_qubits + qoff, gate_m[g], gate_U + uoff, max_terms, min_mass, &kf);
        if (rc != SV_OK) break;
        if (kept_fractions) kept_fractions[g] = kf;
        qoff += gate_m[g]; uoff += (size_t)1 << (2 * gate_m[g]);
        g += 1;
        if (s->small_backoff > 0) s->small_backoff -= 1;
    }
    delete[] h_gates;
    s->circuit_done = g;
    return rc;
}

extern "C" int sv_apply_circuit(sv_state* s, int n_gates, const int* gate_m, const int* gate_qubits, const sv_c128* gate_U,
                                uint64_t max_terms, double min_mass, double* kept_fractions, int* n_done) {
    if (n_done) *n_done = 0;
    if (!s) return SV_ERR_INVALID_ARG;
    if (n_gates < 0 || (n_gates && (!gate_m || !gate_qubits || !gate_U))) return fail(s, SV_ERR_INVALID_ARG, "null argument");
    if (!(min_mass > 0.0)) return fail(s, SV_ERR_INVALID_ARG, "min_mass must be > 0");
    s->err[0] = 0;
    s->circuit_done = 0;
    const int rc = apply_circuit_impl(s, n_gates, gate_m, gate_qubits, gate_U, max_terms, min_mass, kept_fractions);
    if (n_done) *n_done = s->circuit_done;
    return rc;
}

// ---------------------------------------------------------------------------------------
// truncation driver (rows a-8, a-9)
// ---------------------------------------------------------------------------------------
// The exact adaptive radix select over (keys, amps)[0..n).  seeded: the select state has been
// prepared by svk_sel_seed (candidates of the sampled fast path); lk: scratch for tie keys.
static int select_levels(sv_state* s, const u64* keys, const double2* amps, u64 n, u64 n_live, u64* lk, bool seeded, u64 max_terms,
                         double min_mass, SelState* out) {
    const KeyMap km = keymap_of(s);
    if (!seeded) s->stats.launches += svk_sel_init(s->sel, s->hist, n_live, max_terms, min_mass, s->stream, s->pre_valid ? s->pre : nullptr);
    int phase = 0;
    u64 ties = 0;
    {   // The usual course of a select -- exponent level, up to three pattern levels, the tie keys, two key
        // levels -- is launched AHEAD without reading anything back: every pass and step checks on the
        // device that it is the select's current phase and is a no-op otherwise.  One read-back follows.
        cudaEvent_t e0, e1;
        prof_slot(s, SV_K_SELHIST, 16.0 * (double)n, &e0, &e1);
        if (e0) cudaEventRecord(e0, s->stream);
        static const int chain[7] = {0, 1, 1, 1, 2, 3, 3};
        for (int c = 0; c < 7; ++c) {
            const int ph = chain[c];
            if (ph <= 1) s->stats.launches += svk_sel_pass(ph, amps, nullptr, n, s->sel, s->hist, s->stream);
            else if (ph == 2) s->stats.launches += svk_sel_extract(keys, amps, n, s->sel, km, lk, s->hist, s->stream);
            else s->stats.launches += svk_sel_pass(2, nullptr, lk, n, s->sel, s->hist, s->stream);
            s->stats.launches += svk_sel_step(s->sel, s->hist, s->stream, ph);
        }
        if (e1) cudaEventRecord(e1, s->stream);
        CHECK_LAUNCH();
        s->stats.passes += 1;
        int rc = read_back(s, out, s->sel, sizeof(SelState));
        if (rc != SV_OK) return rc;
        if (out->done == 1 || out->done == 3) return SV_OK;
        if (out->done != 0) return fail(s, SV_ERR_CUDA, "internal: radix select inconsistency");
        phase = out->phase;
        ties = out->tie_total;
    }
    for (int it = 0; it < 64; ++it) {
        cudaEvent_t e0, e1;
        const double bytes = phase <= 1 ? 16.0 * (double)n : (phase == 2 ? 16.0 * (double)n + 16.0 * (double)ties : 8.0 * (double)ties);
        prof_slot(s, SV_K_SELHIST, bytes, &e0, &e1);
        if (e0) cudaEventRecord(e0, s->stream);
        if (phase <= 1) s->stats.launches += svk_sel_pass(phase, amps, nullptr, n, s->sel, s->hist, s->stream);
        else if (phase == 2) s->stats.launches += svk_sel_extract(keys, amps, n, s->sel, km, lk, s->hist, s->stream);
        else s->stats.launches += svk_sel_pass(2, nullptr, lk, ties, s->sel, s->hist, s->stream);
        if (e1) cudaEventRecord(e1, s->stream);
        DBG_SYNC(phase <= 1 ? "sel_pass" : (phase == 2 ? "sel_extract" : "sel_pass_keys"));
        s->stats.launches += svk_sel_step(s->sel, s->hist, s->stream);
        DBG_SYNC("sel_step");
        CHECK_LAUNCH();
        s->stats.passes += 1;
        int rc = read_back(s, out, s->sel, sizeof(SelState));
        if (rc != SV_OK) return rc;
        if (out->done == 1 || out->done == 3) return SV_OK;
        if (out->done != 0) return fail(s, SV_ERR_CUDA, "internal: radix select inconsistency");
        phase = out->phase;
        ties = out->tie_total;
    }
    return fail(s, SV_ERR_CUDA, "radix select did not converge");
}

// Sampled fast path (sv_sample_select.cu): one streaming pass over the amplitudes, then the
// exact select on the few candidates around the cut.  *used = false: band miss, nothing decided.
static int run_select_sampled(sv_state* s, u64 max_terms, double min_mass, SelState* out, bool* used) {
    *used = false;
    const u64 n = s->phys, n_live = s->count;   // stored entries (dead ones included) / live terms
    // a band compaction can only follow when the cap will drop more than 1/8 of the stored entries
    const bool want_band = max_terms != 0 && n > max_terms + max_terms / 8;
    const int alt = s->cur ^ 1;
    u64 m64 = n / 8;
    if (m64 > SV_SAMPLE_MAX) m64 = SV_SAMPLE_MAX;
    if (m64 < 64) return SV_OK;
    const u32 M = (u32)m64;
    cudaStream_t st = s->stream;
    // fused diagonal gate + truncate: the gate (and the pending cut) is applied by the classification pass
    const bool xf = s->diag_deferred;
    const PendPred xpd = s->defer;
    s->stats.launches += svk_ss_sample(s->amps[s->cur], n, M, s->smp_k[0], st, s->keys[s->cur], &xpd, xf ? s->tab : nullptr);
    DBG_SYNC("ss_sample");
    int in_alt = 0;
    s->stats.launches += svk_sort_pairs(s->smp_k[0], s->smp_v[0], s->smp_k[1], s->smp_v[1], M, 24, s->smp_scr, st, &in_alt);   // keys are 24-bit pattern prefixes + 1 (< 2^24: finite p)
    const PreCut* pre = s->pre_valid ? s->pre : nullptr;   // outputs the gate's pass left out (fused apply + truncate)
    s->stats.launches += svk_ss_pivot(s->smp_k[in_alt ? 1 : 0], M, n_live, max_terms, min_mass, s->mass_est, s->sctl, st, pre);
    DBG_SYNC("ss_sort+pivot");
    cudaEvent_t e0, e1;
    prof_slot(s, SV_K_CLASSIFY, (xf ? 40.0 : 16.0) * (double)n, &e0, &e1);
    if (e0) cudaEventRecord(e0, st);
    s->stats.launches += svk_ss_classify(s->keys[s->cur], s->amps[s->cur], n, s->sctl, s->keys[alt], s->amps[alt], want_band ? s->seg_cnt : nullptr, st,
                                         s->amps[s->cur], &xpd, xf ? s->tab : nullptr);
    if (e1) cudaEventRecord(e1, st);
    if (xf) { s->diag_deferred = false; s->defer.active = 0; }   // applied in place: dropped terms are dead entries now
    DBG_SYNC("ss_classify");
    s->stats.launches += svk_sel_seed(s->sel, s->hist, s->sctl, n_live, max_terms, min_mass, st, pre);
    DBG_SYNC("sel_seed");
    CHECK_LAUNCH();
    s->stats.passes += 1;
    int rc = read_back(s, out, s->sel, sizeof(SelState));
    if (rc != SV_OK) return rc;
    const u64 cand = out->n_total;
    s->band_above = out->kept_count; s->band_cand = cand;
    if (out->done == 3 || cand > n_live / 2) return SV_OK;   // band miss, or too many candidates to gain anything
    rc = select_levels(s, s->keys[alt], s->amps[alt], cand, cand, s->keys[alt] + cand, true, max_terms, min_mass, out);
    if (rc != SV_OK) return rc;
    if (out->done == 1) { *used = true; s->band_valid = want_band; }
    return SV_OK;
}

static int run_select(sv_state* s, u64 max_terms, double min_mass, SelState* out) {
    s->band_valid = false;
    const u64 n = s->phys;                    // callers have materialised any deferred truncation; dead entries may remain
    if (s->count >= s->sample_min_terms) {
        bool used = false;
        int rc = run_select_sampled(s, max_terms, min_mass, out, &used);
        if (rc != SV_OK || used) return rc;
        s->stats.fallbacks += 1;
    }
    { int rcd = flush_diag(s); if (rcd != SV_OK) return rcd; }   // (a deferred diagonal gate the sampled path did not get to)
    // full-state select; the idle buffer holds the extracted tie keys
    return select_levels(s, s->keys[s->cur], s->amps[s->cur], n, s->count, s->keys[s->cur ^ 1], false, max_terms, min_mass, out);
}

extern "C" int sv_truncate(sv_state* s, uint64_t max_terms, double min_mass, double* kept_fraction) {
    if (!s) return SV_ERR_INVALID_ARG;
    if (!(min_mass > 0.0)) return fail(s, SV_ERR_INVALID_ARG, "min_mass must be > 0");
    s->err[0] = 0;
    s->stats.gate_class = SV_CLASS_NONE; s->stats.m = 0; s->stats.active_bits = 0; s->stats.passes = 0;
    s->stats.n_in = s->count + (s->pre_valid ? s->pre_cnt : 0); s->stats.n_out = s->count;
    if (kept_fraction) *kept_fraction = 1.0;
    const bool needK = max_terms != 0 && max_terms < s->count, needM = min_mass < 1.0;
    if (s->count == 0 || (!needK && !needM)) return SV_OK;
    int rc = SV_OK;
    if (s->defer.active && !s->diag_deferred) rc = materialize(s);   // a second truncation in a row: apply the first one now
    if (rc != SV_OK) return rc;
    DBG_SYNC("before select");
    SelState ss;
    rc = run_select(s, max_terms, min_mass, &ss);
    if (rc != SV_OK) return rc;
    s->mass_est = ss.total_mass;
    if (ss.final_count >= s->count) return SV_OK;   // nothing dropped: bitwise no-op (reading R7)
    s->mass_est = 1.0;                              // renormalised
    // The cut is decided; the compaction + renormalisation is left to the next reader of the
    // state (the next gate's load applies it for free), or to materialize().
    s->defer.active = 1; s->defer.PT = ss.PT; s->defer.KT = ss.KT; s->defer.scale = ss.scale; s->defer.km = keymap_of(s);
    s->count = ss.final_count;
    s->stats.n_out = ss.final_count;
    if (kept_fraction) *kept_fraction = ss.kept_fraction;
    // A cut that drops a large part of the stored entries (the cap after an expanding gate): the entries
    // below the sampled band are squeezed out now, in one scan-free streaming pass, so that the following
    // passes run on a dense array in their position-preserving variants.  The cut proper stays pending
    // (the rejected candidates become dead entries); small cuts ride entirely on the next pass.
    if (s->band_valid && !few_dead(s) && s->phys < (1ull << 32)) {
        const int alt = s->cur ^ 1;
        cudaEvent_t e0, e1;
        prof_slot(s, SV_K_COMPACT, 24.0 * ((double)s->phys + (double)(s->band_above + s->band_cand)), &e0, &e1);
        if (e0) cudaEventRecord(e0, s->stream);
        s->stats.launches += svk_ss_band_compact(s->keys[s->cur], s->amps[s->cur], s->phys, s->sctl, s->seg_cnt, s->chunk_cnt,
                                                 s->status, s->tile_counter, s->keys[alt], s->amps[alt], s->stream);
        if (e1) cudaEventRecord(e1, s->stream);
        CHECK_LAUNCH();
        s->stats.passes += 1;
        s->cur = alt;
        s->phys = s->band_above + s->band_cand;
        s->band_valid = false;
    }
    return SV_OK;
}

extern "C" int sv_norm(sv_state* s, double* mass) {
    if (!s || !mass) return SV_ERR_INVALID_ARG;
    if (s->defer.active) { int rcm = materialize(s); if (rcm != SV_OK) return rcm; }
    s->stats.launches += svk_norm(s->amps[s->cur], s->phys, s->partials, s->d_norm, s->stream);   // dead entries add 0
    CHECK_LAUNCH();
    return read_back(s, mass, s->d_norm, sizeof(double));
}

extern "C" int sv_check_invariants(sv_state* s, int* ok) {
    if (!s || !ok) return SV_ERR_INVALID_ARG;
    const bool was_deferred = s->defer.active != 0;
    { int rcm = materialize(s); if (rcm != SV_OK) return rcm; }
    if (was_deferred) {   // the compaction must have kept exactly the number of terms the select decided
        u64 kept = 0;
        int rck = read_back(s, &kept, s->d_count, sizeof(u64));
        if (rck != SV_OK) return rck;
        if (kept != s->count) { *ok = 0; return SV_OK; }
    }
    s->stats.launches += svk_check(s->keys[s->cur], s->amps[s->cur], s->count, s->n, s->d_bad, s->stream);
    CHECK_LAUNCH();
    int bad = 0;
    int rc = read_back(s, &bad, s->d_bad, sizeof(int));
    if (rc != SV_OK) return rc;
    *ok = (bad == 0 && s->count <= s->cap) ? 1 : 0;
    return SV_OK;
}

// ---------------------------------------------------------------------------------------
// readout (row a-11): select k, gather, order by (p desc, key asc), copy to the host
// ---------------------------------------------------------------------------------------
// `bytes` of scratch inside the idle amplitude buffer, behind its first `keep` bytes; nullptr if they do not fit.
static unsigned char* arena_scratch(sv_state* s, size_t keep, size_t bytes) {
    const size_t room = (size_t)s->cap * 16;
    keep = align_up(keep);
    if (keep > room || bytes > room - keep) return nullptr;
    return reinterpret_cast<unsigned char*>(s->amps[s->cur ^ 1]) + keep;
}
struct TmpBuf {
    void* p = nullptr;
    ~TmpBuf() { if (p) cudaFree(p); }
    int alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 256) == cudaSuccess ? 0 : -1; }
};

extern "C" int sv_top(sv_state* s, uint64_t k, uint64_t* keys, sv_c128* amps, double* probs, uint64_t* n_written) {
    if (!s) return SV_ERR_INVALID_ARG;
    s->err[0] = 0;
    if (s->defer.active) { int rcm = materialize(s); if (rcm != SV_OK) return rcm; }
    const u64 kk = k < s->count ? k : s->count;
    if (n_written) *n_written = kk;
    if (kk == 0) return SV_OK;
    if (kk >= (1ull << 32)) return fail(s, SV_ERR_INVALID_ARG, "sv_top supports k < 2^32");
    SelState ss;
    const int use_sel = kk < s->count;
    if (use_sel) {
        int rc = run_select(s, kk, 1.0, &ss);
        if (rc != SV_OK) return rc;
    }
    const size_t a8 = align_up(kk * 8), a16 = align_up(kk * 16), a4 = align_up(kk * 4);
    const size_t sscr = align_up(svk_sort_scratch_bytes(kk));
    // scratch: the idle amplitude buffer of the arena when the readout fits there (always for a small k), else a
    // temporary allocation (full exports)
    TmpBuf tb;
    const size_t need = a8 * 6 + a16 * 2 + a4 * 2 + sscr;
    unsigned char* b = arena_scratch(s, 0, need);
    if (!b) {
        if (tb.alloc(need) != 0) { cudaGetLastError(); return fail(s, SV_ERR_NOMEM, "sv_top: scratch allocation failed"); }
        b = (unsigned char*)tb.p;
    }
    u64* pat = (u64*)b; b += a8;
    u64* lkey = (u64*)b; b += a8;
    u64* ka = (u64*)b; b += a8;
    u64* kb = (u64*)b; b += a8;
    u64* okey = (u64*)b; b += a8;
    double* oprob = (double*)b; b += a8;
    double2* amp = (double2*)b; b += a16;
    double2* oamp = (double2*)b; b += a16;
    u32* va = (u32*)b; b += a4;
    u32* vb = (u32*)b; b += a4;
    u32* scr = (u32*)b;
    cudaStream_t st = s->stream;
    s->stats.launches += svk_gather_top(s->keys[s->cur], s->amps[s->cur], s->phys, s->sel, use_sel, keymap_of(s), pat, lkey,
                                        amp, s->d_count, kk, st);
    CHECK_LAUNCH();
    u64 got = 0;
    int rc = read_back(s, &got, s->d_count, sizeof(u64));
    if (rc != SV_OK) return rc;
    if (got != kk) return fail(s, SV_ERR_CUDA, "internal: readout selected a different number of terms");
    // order: logical key ascending first, then (stable) ~p ascending = p descending
    CU(cudaMemcpyAsync(ka, lkey, kk * 8, cudaMemcpyDeviceToDevice, st));
    s->stats.launches += svk_iota(va, kk, st);
    int in_alt = 0;
    s->stats.launches += svk_sort_pairs(ka, va, kb, vb, kk, s->n, scr, st, &in_alt);
    u32* perm1 = in_alt ? vb : va;
    u64* k2 = in_alt ? ka : kb;          // the buffer pair not holding perm1 becomes the next input
    u32* v2 = in_alt ? va : vb;
    s->stats.launches += svk_gather_u64(pat, perm1, k2, kk, 1, st);
    CU(cudaMemcpyAsync(v2, perm1, kk * 4, cudaMemcpyDeviceToDevice, st));
    u64* k2alt = in_alt ? kb : ka;
    u32* v2alt = in_alt ? vb : va;
    int in_alt2 = 0;
    s->stats.launches += svk_sort_pairs(k2, v2, k2alt, v2alt, kk, 64, scr, st, &in_alt2);
    u32* perm = in_alt2 ? v2alt : v2;
    s->stats.launches += svk_gather_u64(lkey, perm, okey, kk, 0, st);
    s->stats.launches += svk_gather_c128(amp, perm, oamp, kk, st);
    s->stats.launches += svk_gather_u64(pat, perm, k2, kk, 0, st);   // k2 is free again
    s->stats.launches += svk_pat_to_prob(k2, oprob, kk, st);
    CHECK_LAUNCH();
    if (keys) CU(cudaMemcpyAsync(keys, okey, kk * 8, cudaMemcpyDeviceToHost, st));
    if (amps) CU(cudaMemcpyAsync(amps, oamp, kk * 16, cudaMemcpyDeviceToHost, st));
    if (probs) CU(cudaMemcpyAsync(probs, oprob, kk * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return SV_OK;
}

// ---------------------------------------------------------------------------------------
// load: establish the sorted storage order with the radix sort
// ---------------------------------------------------------------------------------------
// staged: dev_keys / dev_amps live in the arena scratch behind `staged_bytes` of the idle amplitude buffer (sv_load)
static int load_device_impl(sv_state* s, const uint64_t* dev_keys, const sv_c128* dev_amps, uint64_t n, size_t dest_and_staged_bytes) {
    s->err[0] = 0;
    if (n > s->cap) return fail(s, SV_ERR_INVALID_ARG, "sv_load: n exceeds capacity");
    if (n >= (1ull << 32)) return fail(s, SV_ERR_INVALID_ARG, "sv_load supports n < 2^32");
    cudaStream_t st = s->stream;
    const int alt = s->cur ^ 1;
    if (n > 0) {
        const size_t a8 = align_up(n * 8), a4 = align_up(n * 4);
        const size_t need = a8 * 2 + a4 * 2 + align_up(svk_sort_scratch_bytes(n));
        TmpBuf tb;
        unsigned char* b = arena_scratch(s, dest_and_staged_bytes, need);   // behind the destination (and the staged input)
        if (!b) {
            if (tb.alloc(need) != 0) { cudaGetLastError(); return fail(s, SV_ERR_NOMEM, "sv_load: scratch allocation failed"); }
            b = (unsigned char*)tb.p;
        }
        u64* ka = (u64*)b; b += a8;
        u64* kb = (u64*)b; b += a8;
        u32* va = (u32*)b; b += a4;
        u32* vb = (u32*)b; b += a4;
        u32* scr = (u32*)b;
        CU(cudaMemcpyAsync(ka, dev_keys, n * 8, cudaMemcpyDeviceToDevice, st));
        s->stats.launches += svk_iota(va, n, st);
        int in_alt = 0;
        s->stats.launches += svk_sort_pairs(ka, va, kb, vb, n, 64, scr, st, &in_alt);
        CU(cudaMemcpyAsync(s->keys[alt], in_alt ? kb : ka, n * 8, cudaMemcpyDeviceToDevice, st));
        s->stats.launches += svk_gather_c128((const double2*)dev_amps, in_alt ? vb : va, s->amps[alt], n, st);
        s->stats.launches += svk_check(s->keys[alt], s->amps[alt], n, s->n, s->d_bad, st);
        CHECK_LAUNCH();
        int bad = 0;
        int rc = read_back(s, &bad, s->d_bad, sizeof(int));   // (synchronises: a temporary allocation may go now)
        if (rc != SV_OK) return rc;
        if (bad) return fail(s, SV_ERR_INVALID_ARG, "sv_load: duplicate key, key >= 2^n or zero amplitude (state unchanged)");
    }
    s->cur = alt;
    s->count = n; s->phys = n;
    s->defer.active = 0;
    s->lut_valid = false;
    s->mass_est = nan("");
    if (n > 0) {   // the total mass steers the sampled truncation path (it is re-measured exactly there)
        double m = 0.0;
        s->stats.launches += svk_norm(s->amps[s->cur], n, s->partials, s->d_norm, st);
        if (read_back(s, &m, s->d_norm, sizeof(double)) == SV_OK) s->mass_est = m;
    }
    s->xmask = 0;
    for (int q = 0; q < 64; ++q) s->phys_of_log[q] = q;
    s->stats.n_in = n; s->stats.n_out = n; s->stats.gate_class = SV_CLASS_NONE;
    return SV_OK;
}

extern "C" int sv_load_device(sv_state* s, const uint64_t* dev_keys, const sv_c128* dev_amps, uint64_t n) {
    if (!s || (n && (!dev_keys || !dev_amps))) return SV_ERR_INVALID_ARG;
    return load_device_impl(s, dev_keys, dev_amps, n, (size_t)n * 16);
}

extern "C" int sv_load(sv_state* s, const uint64_t* keys, const sv_c128* amps, uint64_t n) {
    if (!s || (n && (!keys || !amps))) return SV_ERR_INVALID_ARG;
    if (n > s->cap) return fail(s, SV_ERR_INVALID_ARG, "sv_load: n exceeds capacity");
    // staging of the host arrays: in the idle amplitude buffer behind the destination when it fits, else temporary
    const size_t a8 = align_up(n * 8), a16 = align_up(n * 16);
    TmpBuf tb;
    size_t behind = a16;
    unsigned char* stg = arena_scratch(s, a16, a8 + a16);
    if (stg) behind = a16 + a8 + a16;
    else {
        if (tb.alloc(a8 + a16) != 0) { cudaGetLastError(); return fail(s, SV_ERR_NOMEM, "sv_load: staging allocation failed"); }
        stg = (unsigned char*)tb.p;
    }
    uint64_t* dk = (uint64_t*)stg;
    sv_c128* da = (sv_c128*)(stg + a8);
    if (n) {
        CU(cudaMemcpyAsync(dk, keys, n * 8, cudaMemcpyHostToDevice, s->stream));
        CU(cudaMemcpyAsync(da, amps, n * 16, cudaMemcpyHostToDevice, s->stream));
    }
    int rc = load_device_impl(s, dk, da, n, behind);
    cudaStreamSynchronize(s->stream);
    return rc;
}

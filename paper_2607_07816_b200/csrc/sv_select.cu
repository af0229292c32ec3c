// Norm, the compaction pass of a truncation (row a-9, also fused with a
// diagonal gate), readout gather and structural checks.  The cut itself is found by the
// radix select in sv_radix_select.cu.
#include "sv_tile.cuh"

// ---------------------------------------------------------------------------------------
// a-10 norm: fixed-order two-stage reduction (deterministic)
// ---------------------------------------------------------------------------------------
#define SV_NORM_BLOCKS 1024
__global__ void __launch_bounds__(SV_THREADS) norm_partial_kernel(const double2* __restrict__ amps, u64 n,
                                                                  double* __restrict__ partials) {
    __shared__ double red[SV_THREADS];
    double s = 0.0;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) s = __dadd_rn(s, prob_of(ld_stream_d2(amps + i)));
    red[threadIdx.x] = s;
    __syncthreads();
    for (int d = SV_THREADS / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) red[threadIdx.x] = __dadd_rn(red[threadIdx.x], red[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = red[0];
}
__global__ void __launch_bounds__(SV_THREADS) norm_final_kernel(const double* __restrict__ partials, int nb,
                                                                double* __restrict__ out) {
    __shared__ double red[SV_THREADS];
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += SV_THREADS) s = __dadd_rn(s, partials[i]);
    red[threadIdx.x] = s;
    __syncthreads();
    for (int d = SV_THREADS / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) red[threadIdx.x] = __dadd_rn(red[threadIdx.x], red[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = red[0];
}
int svk_norm(const double2* amps, u64 n, double* partials, double* d_out, cudaStream_t st) {
    int nb = (int)((n + SV_THREADS * 8 - 1) / (SV_THREADS * 8));
    if (nb < 1) nb = 1;
    if (nb > SV_NORM_BLOCKS) nb = SV_NORM_BLOCKS;
    norm_partial_kernel<<<nb, SV_THREADS, 0, st>>>(amps, n, partials);
    norm_final_kernel<<<1, SV_THREADS, 0, st>>>(partials, nb, d_out);
    return 2;
}

// Number of live entries (amplitude != 0+0i) -> *d_count.  Used after a diagonal gate with exact zeros on its
// diagonal (a projector): the terms it annihilates are dropped, i.e. become dead entries.
__global__ void __launch_bounds__(SV_THREADS) count_live_kernel(const double2* __restrict__ amps, u64 n, u64* d_count) {
    u64 c = 0;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double2 a = ld_stream_d2(amps + i);
        c += (a.x == 0.0 && a.y == 0.0) ? 0 : 1;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(reinterpret_cast<unsigned long long*>(d_count), (unsigned long long)c);
}
// OR and AND of the stored keys of the live entries (a pending truncation applied when with_pend): a stored bit on which
// the two agree has the same value in every term -- the qubit it holds is in a definite state, and bringing it to another
// bit position does not change the order of the keys (sv_api.cu "definite qubits").  out[0] = OR, out[1] = AND.
__global__ void __launch_bounds__(SV_THREADS) key_masks_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps, u64 n,
                                                               PendPred pd, int with_pend, u64* __restrict__ out) {
    u64 o = 0, a = ~0ull;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const u64 k = ld_stream_u64(keys + i);
        bool live = true;
        if (amps) {
            const double2 v = ld_stream_d2(amps + i);
            live = (with_pend && pd.active) ? pend_keep(pd, k, v) : !(v.x == 0.0 && v.y == 0.0);
        }
        if (live) { o |= k; a &= k; }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { o |= __shfl_xor_sync(0xffffffffu, o, d); a &= __shfl_xor_sync(0xffffffffu, a, d); }
    if ((threadIdx.x & 31) == 0) {
        atomicOr(reinterpret_cast<unsigned long long*>(&out[0]), (unsigned long long)o);
        atomicAnd(reinterpret_cast<unsigned long long*>(&out[1]), (unsigned long long)a);
    }
}
int svk_key_masks(const u64* keys, const double2* amps, u64 n, const PendPred& pd, int with_pend, u64* out, cudaStream_t st) {
    const u64 init[2] = {0ull, ~0ull};
    cudaMemcpyAsync(out, init, sizeof(init), cudaMemcpyHostToDevice, st);
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 8 - 1) / (SV_THREADS * 8);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    key_masks_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, pd, with_pend, out);
    return 1;
}
int svk_count_live(const double2* amps, u64 n, u64* d_count, cudaStream_t st) {
    cudaMemsetAsync(d_count, 0, sizeof(u64), st);
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 8 - 1) / (SV_THREADS * 8);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    count_live_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(amps, n, d_count);
    return 1;
}

// ---------------------------------------------------------------------------------------
// a-9 cut + renormalise: stable compaction of the kept prefix, scale fused
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ bool sel_keep(u64 pat, u64 stored_key, u64 PT, u64 KT, const KeyMap& km) {
    if (pat > PT) return true;
    if (pat < PT) return false;
    if (KT == ~0ull) return true;
    return logical_key(stored_key, km) <= KT;
}

#define SV_CMP_IT 8
// DIAG: a diagonal gate (phase table in gtab, see diag_kernel) is applied to the survivors
// in the same pass -- "truncate, then diagonal gate" costs one read and one write.
template <bool DIAG>
__global__ void __launch_bounds__(SV_THREADS) compact_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                             u64* __restrict__ kout, double2* __restrict__ aout, u64 n,
                                                             PendPred pd, const GateTab* __restrict__ gtab,
                                                             u64* status, u32* tile_counter, u64* d_count, u32 ntiles) {
    __shared__ int wcnt[SV_CMP_IT][SV_THREADS / 32];
    __shared__ u32 s_tile;
    __shared__ u64 s_base;
    __shared__ double2 sd[16];
    __shared__ int s_cpos[SV_MAX_M], s_mc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(tile_counter, 1u);
    if (DIAG) {
        if (tid < 16) sd[tid] = gtab->U[tid];
        if (tid < SV_MAX_M) s_cpos[tid] = gtab->ctrl_pos[tid];
        if (tid == 0) s_mc = gtab->mc;
    }
    __syncthreads();
    const u32 tile = s_tile;
    const u64 PT = pd.PT, KT = pd.KT;
    const double scale = pd.active ? pd.scale : 1.0;
    const u64 t0 = (u64)tile * (SV_THREADS * SV_CMP_IT);
    u64 k[SV_CMP_IT]; double2 a[SV_CMP_IT]; u32 ball[SV_CMP_IT];
#pragma unroll
    for (int it = 0; it < SV_CMP_IT; ++it) {
        const u64 i = t0 + (u64)it * SV_THREADS + tid;
        if (i < n) { k[it] = ld_stream_u64(kin + i); a[it] = ld_stream_d2(ain + i); }
        else { k[it] = 0; a[it].x = 0.0; a[it].y = 0.0; }
    }
    int tot = 0;
#pragma unroll
    for (int it = 0; it < SV_CMP_IT; ++it) {
        const u64 i = t0 + (u64)it * SV_THREADS + tid;
        bool keep = false;
        if (i < n && !(a[it].x == 0.0 && a[it].y == 0.0))   // dead entries (0+0i) are squeezed out
            keep = !pd.active || sel_keep((u64)__double_as_longlong(prob_of(a[it])), k[it], PT, KT, pd.km);
        const u32 b = __ballot_sync(0xffffffffu, keep);
        ball[it] = b;
        if (lane == 0) wcnt[it][warp] = __popc(b);
    }
    __syncthreads();
    if (tid < 32) {   // exclusive offsets of the IT x 8 warp counts (one per lane pair), tile total, look-back
        int c0 = 0, c1 = 0;
        const int e0 = 2 * lane, e1 = 2 * lane + 1;   // 64 entries, row-major [it][warp]
        c0 = wcnt[e0 >> 3][e0 & 7]; c1 = wcnt[e1 >> 3][e1 & 7];
        int inc = c0 + c1;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
        tot = __shfl_sync(0xffffffffu, inc, 31);
        const int ex = inc - c0 - c1;
        __syncwarp();
        wcnt[e0 >> 3][e0 & 7] = ex; wcnt[e1 >> 3][e1 & 7] = ex + c0;
        const u64 excl = lookback_exclusive_2level(status, status + ntiles, tile, ntiles, (u64)tot);
        if (lane == 0) { s_base = excl; if (tile == ntiles - 1) *d_count = excl + (u64)tot; }
    }
    __syncthreads();
    const u64 base = s_base;
    const int mc = DIAG ? s_mc : 0;
#pragma unroll
    for (int it = 0; it < SV_CMP_IT; ++it) {
        if ((ball[it] >> lane) & 1u) {
            const u64 pos = base + (u64)wcnt[it][warp] + (u64)__popc(ball[it] & ((1u << lane) - 1u));
            st_stream_u64(kout + pos, k[it]);
            double2 o; o.x = __dmul_rn(a[it].x, scale); o.y = __dmul_rn(a[it].y, scale);
            if (DIAG) {
                int cx = 0;
                for (int j = 0; j < mc; ++j) cx |= (int)((k[it] >> s_cpos[j]) & 1ull) << j;
                const double2 u = sd[cx];
                double2 r;
                r.x = __dsub_rn(__dmul_rn(u.x, o.x), __dmul_rn(u.y, o.y));
                r.y = __dadd_rn(__dmul_rn(u.x, o.y), __dmul_rn(u.y, o.x));
                o = r;
            }
            st_stream_d2(aout + pos, o);
        }
    }
}

static int launch_compact(bool diag, const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, const PendPred& pd,
                          const GateTab* tab, u64* status, u32* tile_counter, u64* d_count, cudaStream_t st) {
    if (n == 0) return 0;
    const u32 ntiles = (u32)((n + SV_THREADS * SV_CMP_IT - 1) / (SV_THREADS * SV_CMP_IT));
    cudaMemsetAsync(status, 0, ((size_t)ntiles + (ntiles + 31) / 32 + 8) * sizeof(u64), st);   // tile + group statuses
    cudaMemsetAsync(tile_counter, 0, sizeof(u32), st);
    if (diag) compact_kernel<true><<<ntiles, SV_THREADS, 0, st>>>(kin, ain, kout, aout, n, pd, tab, status, tile_counter, d_count, ntiles);
    else compact_kernel<false><<<ntiles, SV_THREADS, 0, st>>>(kin, ain, kout, aout, n, pd, tab, status, tile_counter, d_count, ntiles);
    return 1;
}
int svk_compact(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, const PendPred& pd, u64* status,
                u32* tile_counter, u64* d_count, cudaStream_t st) {
    return launch_compact(false, kin, ain, kout, aout, n, pd, nullptr, status, tile_counter, d_count, st);
}
int svk_diag_compact(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, const GateTab* tab,
                     const PendPred& pend, u64* status, u32* tile_counter, u64* d_count, cudaStream_t st) {
    return launch_compact(true, kin, ain, kout, aout, n, pend, tab, status, tile_counter, d_count, st);
}

// Diagonal gate fused with a pending truncation, IN PLACE: survivors are scaled and multiplied by
// their phase, dropped terms become dead entries (0+0i) that later passes skip or squeeze out.
// 40 B per term (key read, amplitude read + write), no scan.
__global__ void __launch_bounds__(SV_THREADS) diag_pend_kernel(const u64* __restrict__ keys, double2* __restrict__ amps, u64 n,
                                                               PendPred pd, const GateTab* __restrict__ gtab, int has_phase) {
    __shared__ double2 sd[16];
    __shared__ int s_cpos[SV_MAX_M], s_mc;
    if (threadIdx.x < 16) sd[threadIdx.x] = gtab->U[threadIdx.x];
    if (threadIdx.x < SV_MAX_M) s_cpos[threadIdx.x] = gtab->ctrl_pos[threadIdx.x];
    if (threadIdx.x == 0) s_mc = gtab->mc;
    __syncthreads();
    const int mc = has_phase ? s_mc : 0;
    const u64 PT = pd.PT, KT = pd.KT;
    const double scale = pd.scale;
    const u64 chunk = (u64)SV_THREADS * 4;
    const u64 nchunks = (n + chunk - 1) / chunk;
    for (u64 c = blockIdx.x; c < nchunks; c += gridDim.x) {
        u64 k[4]; double2 a[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            k[r] = 0; a[r] = make_double2(0.0, 0.0);
            if (i < n) { k[r] = ld_stream_u64(keys + i); a[r] = amps[i]; }
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            if (i >= n || (a[r].x == 0.0 && a[r].y == 0.0)) continue;   // dead stays dead (nothing to write)
            double2 o = make_double2(0.0, 0.0);
            if (sel_keep((u64)__double_as_longlong(prob_of(a[r])), k[r], PT, KT, pd.km)) {
                o.x = __dmul_rn(a[r].x, scale); o.y = __dmul_rn(a[r].y, scale);
                if (has_phase) {
                    int cx = 0;
                    for (int j = 0; j < mc; ++j) cx |= (int)((k[r] >> s_cpos[j]) & 1ull) << j;
                    const double2 u = sd[cx];
                    double2 t;
                    t.x = __dsub_rn(__dmul_rn(u.x, o.x), __dmul_rn(u.y, o.y));
                    t.y = __dadd_rn(__dmul_rn(u.x, o.y), __dmul_rn(u.y, o.x));
                    o = t;
                }
            }
            amps[i] = o;
        }
    }
}
int svk_diag_pend(const u64* keys, double2* amps, u64 n, const GateTab* tab, int has_phase, const PendPred& pend, cudaStream_t st) {
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    diag_pend_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, pend, tab, has_phase);
    return 1;
}

// ---------------------------------------------------------------------------------------
// readout support: gather the selected terms as (p pattern, logical key, amplitude)
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SV_THREADS) gather_top_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps,
                                                                u64 n, const SelState* __restrict__ ssp, int use_sel,
                                                                KeyMap km, u64* __restrict__ o_pat, u64* __restrict__ o_lkey,
                                                                double2* __restrict__ o_amp, u64* d_count, u64 kmax) {
    const u64 PT = use_sel ? ssp->PT : 0, KT = use_sel ? ssp->KT : ~0ull;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const u64 k = keys[i];
        const double2 a = amps[i];
        const u64 pat = (u64)__double_as_longlong(prob_of(a));
        if (a.x == 0.0 && a.y == 0.0) continue;   // dead entry
        if (!use_sel || sel_keep(pat, k, PT, KT, km)) {
            const u64 pos = atomicAdd(d_count, 1ull);
            if (pos < kmax) { o_pat[pos] = pat; o_lkey[pos] = logical_key(k, km); o_amp[pos] = a; }
        }
    }
}
int svk_gather_top(const u64* keys, const double2* amps, u64 n, const SelState* ss, int use_sel, KeyMap km, u64* o_pat,
                   u64* o_lkey, double2* o_amp, u64* d_count, u64 kmax, cudaStream_t st) {
    cudaMemsetAsync(d_count, 0, sizeof(u64), st);
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    gather_top_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, ss, use_sel, km, o_pat, o_lkey, o_amp,
                                                               d_count, kmax);
    return 1;
}

// ---------------------------------------------------------------------------------------
// structural invariants (tests): strictly ascending stored keys, keys < 2^n, no exact zero
// ---------------------------------------------------------------------------------------
__global__ void check_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps, u64 n, int nq, int* bad) {
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const u64 k = keys[i];
        const double2 a = amps[i];
        bool b = false;
        if (i > 0 && keys[i - 1] >= k) b = true;
        if (nq < 64 && (k >> nq) != 0) b = true;
        if (a.x == 0.0 && a.y == 0.0) b = true;   // callers compact dead entries away first
        if (b) atomicExch(bad, 1);
    }
}
int svk_check(const u64* keys, const double2* amps, u64 n, int nq, int* d_bad, cudaStream_t st) {
    cudaMemsetAsync(d_bad, 0, sizeof(int), st);
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    check_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, nq, d_bad);
    return 1;
}

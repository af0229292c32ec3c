// Truncation, norm (a-10) and structural checks.
//
// PAPER.md:124 sorts the terms by probability and cuts a prefix.  Here the cut is found
// without sorting: a most-significant-digit radix SELECT over the 64-bit patterns of
// p = re*re + im*im (monotone as unsigned integers for p >= 0), 12 bits per level, that
// carries per-bin term counts AND exact per-bin masses, so the top-k cut and the p-mass
// cut fall out of the same histograms.  Ties at the cutoff probability
// are resolved by a second select on the logical key, ascending.  One stable compaction
// pass then keeps the prefix and multiplies by 1/sqrt(kept mass).
//
// Exact masses: inside one bin all probabilities share the exponent E, so the bin's mass
// is 2^(E-1075) * sum(M), M the 53-bit significand; sum(M) is kept as two integer sums
// (M >> 26 and M & (2^26 - 1)) which cannot overflow 64 bits.  Integer sums are order
// independent, so every run gives bit-identical cut decisions (D3).
#include "sv_device.cuh"

// ---------------------------------------------------------------------------------------
// double-double helpers (cut decisions only; one thread)
// ---------------------------------------------------------------------------------------
struct dd { double hi, lo; };
__device__ __forceinline__ dd dd_make(double a) { dd r; r.hi = a; r.lo = 0.0; return r; }
__device__ __forceinline__ dd two_sum(double a, double b) {
    dd r; r.hi = __dadd_rn(a, b);
    const double bb = __dsub_rn(r.hi, a);
    r.lo = __dadd_rn(__dsub_rn(a, __dsub_rn(r.hi, bb)), __dsub_rn(b, bb));
    return r;
}
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    s.lo = __dadd_rn(s.lo, __dadd_rn(a.lo, b.lo));
    return two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { b.hi = -b.hi; b.lo = -b.lo; return dd_add(a, b); }
__device__ __forceinline__ bool dd_ge(dd a, dd b) { return a.hi > b.hi || (a.hi == b.hi && a.lo >= b.lo); }
__device__ __forceinline__ dd dd_from_u64(u64 x) {
    return two_sum(__dmul_rn((double)(x >> 32), 4294967296.0), (double)(x & 0xffffffffull));
}
__device__ __forceinline__ dd dd_scale2(dd a, int e) { a.hi = ldexp(a.hi, e); a.lo = ldexp(a.lo, e); return a; }
// mass of a bin: (shi * 2^26 + slo) * 2^(E - 1075)
__device__ __forceinline__ dd bin_mass(u64 shi, u64 slo, int E) {
    dd h = dd_scale2(dd_from_u64(shi), 26);
    return dd_scale2(dd_add(h, dd_from_u64(slo)), E - 1075);
}

__device__ __forceinline__ int p_shift(int level) { return level < 5 ? 52 - 12 * level : 0; }
__device__ __forceinline__ int p_bits(int level) { return level < 5 ? 12 : 4; }
// key level kl covers logical key bits [lo, top)
__device__ __forceinline__ int k_top(int nq, int kl) { return nq - 12 * kl; }
__device__ __forceinline__ int k_lo(int nq, int kl) { int t = nq - 12 * kl - 12; return t < 0 ? 0 : t; }

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

// ---------------------------------------------------------------------------------------
// select: state init, per-level histogram, per-level decision
// ---------------------------------------------------------------------------------------
__global__ void sel_init_kernel(SelState* ss, u64 n, u64 max_terms, double min_mass) {
    SelState s;
    memset(&s, 0, sizeof(s));
    s.n_total = n;
    s.count_active = (max_terms != 0 && max_terms < n) ? 1 : 0;
    s.k_rem = max_terms;
    s.mass_active = (min_mass < 1.0) ? 1 : 0;
    s.mass_rem_hi = min_mass;   // turned into min_mass * S once S is known (level 0)
    s.cand_count = n;
    *ss = s;
}
int svk_sel_init(SelState* ss, u64 n, u64 max_terms, double min_mass, cudaStream_t st) {
    sel_init_kernel<<<1, 1, 0, st>>>(ss, n, max_terms, min_mass);
    return 1;
}

// hist layout: [0..4096) counts, [4096..8192) sum(M >> 26), [8192..12288) sum(M & (2^26-1))
__global__ void __launch_bounds__(SV_THREADS) sel_hist_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps,
                                                              u64 n, const SelState* __restrict__ ssp, KeyMap km, int nq,
                                                              u64* __restrict__ hist) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* shi = reinterpret_cast<u64*>(smem_raw);
    u64* slo = shi + SV_SEL_BINS;
    u32* scnt = reinterpret_cast<u32*>(slo + SV_SEL_BINS);
    for (int i = threadIdx.x; i < SV_SEL_BINS; i += SV_THREADS) { shi[i] = 0; slo[i] = 0; scnt[i] = 0; }
    __syncthreads();
    const int level = ssp->level;
    const u64 pprefix = ssp->pat_prefix, kprefix = ssp->key_prefix;
    const bool keyphase = level >= 6;
    const int shift = keyphase ? k_lo(nq, level - 6) : p_shift(level);
    const int bits = keyphase ? (k_top(nq, level - 6) - k_lo(nq, level - 6)) : p_bits(level);
    const int top = shift + bits;
    const u32 dmask = (1u << bits) - 1u;
    const int lane = threadIdx.x & 31;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    const u64 nround = (n + stride - 1) / stride;
    for (u64 it = 0; it < nround; ++it) {
        const u64 i = it * stride + (u64)blockIdx.x * blockDim.x + threadIdx.x;
        bool valid = i < n;
        u64 pat = 0;
        if (valid) pat = (u64)__double_as_longlong(prob_of(ld_stream_d2(amps + i)));
        u32 bin = 0;
        if (!keyphase) {
            if (valid && level > 0) valid = (pat >> top) == pprefix;
            bin = (u32)(pat >> shift) & dmask;
        } else {
            valid = valid && (pat == pprefix);
            if (valid) {
                const u64 lk = logical_key(keys[i], km);
                if (top < 64 && (lk >> top) != kprefix) valid = false;
                bin = (u32)(lk >> shift) & dmask;
            }
        }
        const u64 mant = pat & ((1ull << 52) - 1);
        const u64 M = ((pat >> 52) & 0x7ff) ? (mant | (1ull << 52)) : mant;
        u64 h = M >> 26, l = M & ((1ull << 26) - 1);
        if (level == 0) {
            // few distinct exponent bins per warp: aggregate per bin before touching smem
            u32 todo = __ballot_sync(0xffffffffu, valid);
            while (todo) {
                const int ldr = __ffs(todo) - 1;
                const u32 b0 = __shfl_sync(0xffffffffu, bin, ldr);
                const bool mine = valid && bin == b0;
                const u32 grp = __ballot_sync(0xffffffffu, mine);
                u64 hh = mine ? h : 0, ll = mine ? l : 0;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) {
                    hh += __shfl_xor_sync(0xffffffffu, hh, d);
                    ll += __shfl_xor_sync(0xffffffffu, ll, d);
                }
                if (lane == ldr) {
                    atomicAdd(&scnt[b0], (u32)__popc(grp));
                    atomicAdd(&shi[b0], hh);
                    atomicAdd(&slo[b0], ll);
                }
                todo &= ~grp;
            }
        } else if (valid) {
            atomicAdd(&scnt[bin], 1u);
            if (!keyphase) { atomicAdd(&shi[bin], h); atomicAdd(&slo[bin], l); }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < SV_SEL_BINS; i += SV_THREADS) {
        const u32 c = scnt[i];
        if (c) {
            atomicAdd(&hist[i], (u64)c);
            if (!keyphase) { atomicAdd(&hist[SV_SEL_BINS + i], shi[i]); atomicAdd(&hist[2 * SV_SEL_BINS + i], slo[i]); }
        }
    }
}

int svk_sel_hist(const u64* keys, const double2* amps, u64 n, const SelState* ss, KeyMap km, int nq, u64* hist,
                 cudaStream_t st) {
    const size_t smem = (size_t)SV_SEL_BINS * (8 + 8 + 4);
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(sel_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr = true; }
    u64 blocks = (n + SV_THREADS * 8 - 1) / (SV_THREADS * 8);
    if (blocks > 148 * 2) blocks = 148 * 2;
    if (blocks < 1) blocks = 1;
    sel_hist_kernel<<<(unsigned)blocks, SV_THREADS, smem, st>>>(keys, amps, n, ss, km, nq, hist);
    return 1;
}

// One decision step: reads the level's histogram, narrows the cut to one bin (or finishes),
// and clears the histogram for the next level.  One block; thread 0 decides.
__global__ void __launch_bounds__(SV_THREADS) sel_step_kernel(SelState* ssp, u64* hist, int nq) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* h = reinterpret_cast<u64*>(smem_raw);   // 3 * 4096
    for (int i = threadIdx.x; i < 3 * SV_SEL_BINS; i += SV_THREADS) { h[i] = hist[i]; hist[i] = 0; }
    __syncthreads();
    if (threadIdx.x != 0) return;
    SelState s = *ssp;
    const u64* cnt = h;
    const u64* shi = h + SV_SEL_BINS;
    const u64* slo = h + 2 * SV_SEL_BINS;
    dd kept; kept.hi = s.kept_hi; kept.lo = s.kept_lo;
    dd rem; rem.hi = s.mass_rem_hi; rem.lo = s.mass_rem_lo;
    if (s.level < 6) {
        const int level = s.level, bits = p_bits(level), nb = 1 << bits;
        int E = 0;
        if (level > 0) { const int ef = (int)((s.pat_prefix >> (12 * level - 12)) & 0x7ff); E = ef ? ef : 1; }
        if (level == 0) {   // total mass S, and the p-mass threshold min_mass * S  (reading R5)
            dd tot = dd_make(0.0);
            for (int d = 0; d < nb; ++d)
                if (cnt[d]) tot = dd_add(tot, bin_mass(shi[d], slo[d], (d & 0x7ff) ? (d & 0x7ff) : 1));
            s.total_hi = tot.hi; s.total_lo = tot.lo;
            rem = dd_make(__dmul_rn(s.mass_rem_hi, tot.hi));
        }
        u64 cumc = 0; dd cum = dd_make(0.0);
        int dK = -1, dM = -1, dlow = -1;
        u64 aboveC_K = 0, aboveC_M = 0; dd aboveM_K = dd_make(0.0), aboveM_M = dd_make(0.0);
        for (int d = nb - 1; d >= 0; --d) {
            const u64 c = cnt[d];
            if (!c) continue;
            dlow = d;
            const dd m = bin_mass(shi[d], slo[d], level == 0 ? ((d & 0x7ff) ? (d & 0x7ff) : 1) : E);
            if (s.count_active && dK < 0 && cumc + c >= s.k_rem) { dK = d; aboveC_K = cumc; aboveM_K = cum; }
            if (s.mass_active && dM < 0 && dd_ge(dd_add(cum, m), rem)) { dM = d; aboveC_M = cumc; aboveM_M = cum; }
            if ((dK >= 0 || !s.count_active) && (dM >= 0 || !s.mass_active)) break;
            cumc += c; cum = dd_add(cum, m);
        }
        // threshold never reached (rounding of min_mass * S): everything is needed
        if (s.mass_active && dM < 0) { dM = dlow; aboveC_M = cumc - cnt[dlow]; aboveM_M = dd_sub(cum, bin_mass(shi[dlow], slo[dlow], level == 0 ? ((dlow & 0x7ff) ? (dlow & 0x7ff) : 1) : E)); rem = dd_add(cum, dd_make(0.0)); }
        if (s.count_active && dK < 0) { dK = dlow; aboveC_K = cumc - cnt[dlow]; aboveM_K = dd_sub(cum, bin_mass(shi[dlow], slo[dlow], level == 0 ? ((dlow & 0x7ff) ? (dlow & 0x7ff) : 1) : E)); s.k_rem = cumc; }
        int dcut; u64 aboveC; dd aboveM;
        if (s.count_active && s.mass_active) {
            if (dK > dM) s.mass_active = 0; else if (dM > dK) s.count_active = 0;
        }
        if (s.count_active) { dcut = dK; aboveC = aboveC_K; aboveM = aboveM_K; }
        else { dcut = dM; aboveC = aboveC_M; aboveM = aboveM_M; }
        s.kept_count += aboveC; kept = dd_add(kept, aboveM);
        if (s.count_active) s.k_rem -= aboveC;
        if (s.mass_active) rem = dd_sub(rem, aboveM);
        s.pat_prefix = (s.pat_prefix << bits) | (u64)dcut;
        s.cand_count = cnt[dcut];
        const int Ecut = level == 0 ? ((dcut & 0x7ff) ? (dcut & 0x7ff) : 1) : E;
        const dd bm = bin_mass(shi[dcut], slo[dcut], Ecut);
        bool take_all = false;
        if (s.cand_count == 1) take_all = true;
        else {
            const bool allK = !s.count_active || s.k_rem >= s.cand_count;
            if (!s.mass_active && allK) take_all = true;
            else if (s.mass_active && allK) s.count_active = 0;
        }
        const int shift = p_shift(level);
        if (take_all) {
            s.PT = s.pat_prefix << shift; s.KT = ~0ull;
            s.kept_count += s.cand_count; kept = dd_add(kept, bm);
            s.done = 1;
        } else if (level == 5) {   // exact probability reached: the candidates are ties
            const double pv = __longlong_as_double((long long)s.pat_prefix);
            u64 t = s.cand_count;
            if (s.count_active && s.k_rem < t) t = s.k_rem;
            if (s.mass_active) {
                // smallest tm with tm * pv >= rem
                double qd = ceil(rem.hi / pv);
                u64 tm = qd < 1.0 ? 1 : (qd > 1.8e19 ? s.cand_count : (u64)qd);
                if (tm > s.cand_count) tm = s.cand_count;
                // fix rounding of the quotient with an exact product check
                while (tm > 1) { dd pr = two_sum(__dmul_rn((double)(tm - 1), pv), __fma_rn((double)(tm - 1), pv, -__dmul_rn((double)(tm - 1), pv))); if (dd_ge(pr, rem)) --tm; else break; }
                while (tm < s.cand_count) { dd pr = two_sum(__dmul_rn((double)tm, pv), __fma_rn((double)tm, pv, -__dmul_rn((double)tm, pv))); if (!dd_ge(pr, rem)) ++tm; else break; }
                if (tm < t) t = tm;
            }
            if (t < 1) t = 1;
            s.PT = s.pat_prefix;
            const dd tmass = two_sum(__dmul_rn((double)t, pv), __fma_rn((double)t, pv, -__dmul_rn((double)t, pv)));
            kept = dd_add(kept, tmass);          // t tied terms of probability pv are kept in any case
            if (t >= s.cand_count) { s.KT = ~0ull; s.kept_count += s.cand_count; s.done = 1; }
            else { s.k_rem = t; s.count_active = 1; s.mass_active = 0; s.level = 6; s.key_prefix = 0; }
        }
        if (!s.done && s.level < 6 && level < 5) s.level = level + 1;
    } else {
        const int kl = s.level - 6;
        const int lo = k_lo(nq, kl), bits = k_top(nq, kl) - lo, nb = 1 << bits;
        u64 cumc = 0; int dcut = nb - 1;
        for (int d = 0; d < nb; ++d) {
            if (cumc + cnt[d] >= s.k_rem) { dcut = d; break; }
            cumc += cnt[d];
        }
        s.kept_count += cumc; s.k_rem -= cumc;
        s.key_prefix = (s.key_prefix << bits) | (u64)dcut;
        s.cand_count = cnt[dcut];
        if (s.k_rem >= s.cand_count || lo == 0) {
            s.KT = (lo == 0) ? s.key_prefix : ((s.key_prefix << lo) | ((1ull << lo) - 1));
            s.kept_count += s.cand_count;
            s.done = 1;
        } else s.level += 1;
    }
    s.kept_hi = kept.hi; s.kept_lo = kept.lo;
    s.mass_rem_hi = rem.hi; s.mass_rem_lo = rem.lo;
    if (s.done) {
        s.kept_mass = kept.hi; s.total_mass = s.total_hi;
        s.scale = __ddiv_rn(1.0, __dsqrt_rn(s.kept_mass));
        s.kept_fraction = __ddiv_rn(s.kept_mass, s.total_mass);
        s.final_count = s.kept_count;
    }
    *ssp = s;
}
int svk_sel_step(SelState* ss, u64* hist, int nq, cudaStream_t st) {
    const size_t smem = (size_t)3 * SV_SEL_BINS * 8;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(sel_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr = true; }
    sel_step_kernel<<<1, SV_THREADS, smem, st>>>(ss, hist, nq);
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
    const double scale = pd.scale;
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
        if (i < n) keep = sel_keep((u64)__double_as_longlong(prob_of(a[it])), k[it], PT, KT, pd.km);
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
        const u64 excl = lookback_exclusive_warp(status, tile, (u64)tot);
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
    cudaMemsetAsync(status, 0, (size_t)ntiles * sizeof(u64), st);
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
    if (blocks > 148 * 8) blocks = 148 * 8;
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
        if (a.x == 0.0 && a.y == 0.0) b = true;
        if (b) atomicExch(bad, 1);
    }
}
int svk_check(const u64* keys, const double2* amps, u64 n, int nq, int* d_bad, cudaStream_t st) {
    cudaMemsetAsync(d_bad, 0, sizeof(int), st);
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > 148 * 8) blocks = 148 * 8;
    check_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, nq, d_bad);
    return 1;
}

// Truncation cut: where PAPER.md:124 sorts all terms by probability, this
// finds the cut of the (p desc, key asc) order with an ADAPTIVE most-significant-digit radix
// select over the 64-bit patterns of p = re*re + im*im (monotone as unsigned integers).
//
//   level 0      digit = sign + exponent field (2048 bins)
//   later levels digit = the 11 most significant bits in which the candidates of the cut
//                bin still DIFFER.  Every pass keeps, per bin, the AND and the OR of its
//                members' patterns, so the bits that are common to all candidates are
//                resolved for free.  A state full of exact ties (Clifford-like circuits)
//                needs 2 levels instead of 6; distinct values shrink by 2048x per level.
//   ties         if the cut falls inside a group of equal probabilities, the logical keys
//                of that group are extracted once (8 B each) and the same adaptive select
//                runs on them, ascending (reading R4).
//
// Every pass carries per-bin term counts AND exact per-bin masses, so the top-k cut and the
// p-mass cut fall out of the same histograms.  Exact masses: inside one
// bin all probabilities share the exponent E, so the bin's mass is 2^(E-1075) * sum(M), M
// the 53-bit significand; sum(M) is kept as two integer sums (M >> 26, M & (2^26-1)) that
// cannot overflow.  Integer sums are order independent: every run takes bit-identical
// decisions (D3).  The decisions are taken by one thread in double-double.
#include "sv_device.cuh"
#include "sv_launch.cuh"

// ---------------------------------------------------------------------------------------
// double-double helpers (cut decisions only; one thread)
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ dd dd_from_u64(u64 x) {
    return two_sum(__dmul_rn((double)(x >> 32), 4294967296.0), (double)(x & 0xffffffffull));
}
__device__ __forceinline__ dd dd_scale2(dd a, int e) { a.hi = ldexp(a.hi, e); a.lo = ldexp(a.lo, e); return a; }
// mass of a bin: (shi * 2^26 + slo) * 2^(E - 1075)
__device__ __forceinline__ dd bin_mass(u64 shi, u64 slo, int E) {
    dd h = dd_scale2(dd_from_u64(shi), 26);
    return dd_scale2(dd_add(h, dd_from_u64(slo)), E - 1075);
}


#define RS_BINS 2048
// global histogram layout (u64 each): cnt | shi | slo | band | bor | 3 extraction scalars
#define H_CNT 0
#define H_SHI (RS_BINS)
#define H_SLO (2 * RS_BINS)
#define H_AND (3 * RS_BINS)
#define H_OR  (4 * RS_BINS)
#define H_EXT (5 * RS_BINS)     // [0] = extracted count, [1] = AND of the keys, [2] = OR of the keys
#define H_TOTAL (5 * RS_BINS + 8)

// bits of v at the positions of mask, most significant first (order preserving digit)
__device__ __forceinline__ u32 pext_desc(u64 v, u64 mask) {
    u32 r = 0;
    while (mask) {
        const int b = 63 - __clzll((long long)mask);
        r = (r << 1) | (u32)((v >> b) & 1ull);
        mask &= ~(1ull << b);
    }
    return r;
}
__device__ __forceinline__ u64 pdep_desc(u32 d, u64 mask) {
    const int nb = __popcll(mask);
    u64 out = 0;
    int i = nb - 1;
    while (mask) {
        const int b = 63 - __clzll((long long)mask);
        if ((d >> i) & 1u) out |= 1ull << b;
        mask &= ~(1ull << b);
        --i;
    }
    return out;
}
__device__ __forceinline__ u64 top_bits(u64 diff, int k) {   // the k most significant set bits of diff
    u64 m = 0;
    while (diff && k > 0) {
        const int b = 63 - __clzll((long long)diff);
        m |= 1ull << b; diff &= ~(1ull << b); --k;
    }
    return m;
}

__global__ void sel_init_kernel(SelState* ss, u64* hist, u64 n, u64 max_terms, double min_mass, const PreCut* pre) {
    for (int i = threadIdx.x; i < H_TOTAL; i += blockDim.x)
        hist[i] = ((i >= H_AND && i < H_OR) || i == H_EXT + 1) ? ~0ull : 0ull;
    if (threadIdx.x == 0) {
        SelState s;
        memset(&s, 0, sizeof(s));
        s.n_total = n;
        s.count_active = (max_terms != 0 && max_terms < n) ? 1 : 0;
        s.k_rem = max_terms;
        s.mass_active = (min_mass < 1.0) ? 1 : 0;
        s.min_mass = min_mass;
        s.cand_count = n;
        if (pre) { s.pre_hi = pre->mass_hi; s.pre_lo = pre->mass_lo; }   // left out by a fused apply + truncate: part of S
        *ss = s;
    }
}
int svk_sel_init(SelState* ss, u64* hist, u64 n, u64 max_terms, double min_mass, cudaStream_t st, const PreCut* pre) {
    sel_init_kernel<<<1, SV_THREADS, 0, st>>>(ss, hist, n, max_terms, min_mass, pre);
    return 1;
}

// One histogram pass.  MODE 0: exponent level over the amplitudes; MODE 1: adaptive pattern
// level over the amplitudes; MODE 2: adaptive key level over the extracted logical keys.
#define SP_IT 4
template <int MODE>
__global__ void __launch_bounds__(SV_THREADS) sel_pass_kernel(const double2* __restrict__ amps, const u64* __restrict__ lkeys,
                                                              u64 n, const SelState* __restrict__ ssp, u64* __restrict__ hist) {
    // Launched ahead of the decision steps (see select_levels): a pass whose level is not the select's
    // current phase, or that comes after the cut is final, does nothing.
    if (ssp->done != 0 || ssp->phase != (MODE == 0 ? 0 : (MODE == 1 ? 1 : 3))) return;
    if (MODE == 2 && ssp->tie_total < n) n = ssp->tie_total;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u32* scnt = reinterpret_cast<u32*>(smem_raw);
    u32* sand_lo = scnt + RS_BINS;
    u32* sand_hi = sand_lo + RS_BINS;
    u32* sor_lo = sand_hi + RS_BINS;
    u32* sor_hi = sor_lo + RS_BINS;
    u64* shi = reinterpret_cast<u64*>(sor_hi + RS_BINS);   // MODE < 2 only
    u64* slo = shi + RS_BINS;
    for (int i = threadIdx.x; i < RS_BINS; i += SV_THREADS) {
        scnt[i] = 0; sand_lo[i] = ~0u; sand_hi[i] = ~0u; sor_lo[i] = 0; sor_hi[i] = 0;
        if (MODE < 2) { shi[i] = 0; slo[i] = 0; }
    }
    __syncthreads();
    const u64 rmask = MODE == 1 ? ssp->rmask : (MODE == 2 ? ssp->krmask : 0);
    const u64 rval = MODE == 1 ? ssp->rval : (MODE == 2 ? ssp->krval : 0);
    const u64 dmask = MODE == 1 ? ssp->dmask : (MODE == 2 ? ssp->kdmask : 0);
    const int lane = threadIdx.x & 31;
    const u64 chunk = (u64)SV_THREADS * SP_IT;
    const u64 nchunks = (n + chunk - 1) / chunk;
    for (u64 c = blockIdx.x; c < nchunks; c += gridDim.x) {
        u64 v[SP_IT];
        bool ok[SP_IT];
#pragma unroll
        for (int r = 0; r < SP_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            ok[r] = i < n;
            v[r] = 0;
            if (ok[r]) {
                if (MODE == 2) v[r] = ld_stream_u64(lkeys + i);
                else {
                    const double2 a = ld_stream_d2(amps + i);
                    v[r] = (u64)__double_as_longlong(prob_of(a));
                    if (a.x == 0.0 && a.y == 0.0) ok[r] = false;   // dead entry
                }
            }
        }
#pragma unroll
        for (int r = 0; r < SP_IT; ++r) {
            const u64 x = v[r];
            bool valid = ok[r];
            u32 bin;
            if (MODE == 0) bin = (u32)(x >> 52) & (RS_BINS - 1);   // (p >= 0: the sign bit is clear)
            else { valid = valid && ((x & rmask) == rval); bin = valid ? pext_desc(x, dmask) : 0; }
            const u64 mant = x & ((1ull << 52) - 1);
            const u64 M = ((x >> 52) & 0x7ff) ? (mant | (1ull << 52)) : mant;
            const u32 h = (u32)(M >> 26), l = (u32)(M & ((1ull << 26) - 1));
            // lanes of the warp that hit the same bin form a group (one match instruction); the group's sums, AND and
            // OR are reduced inside the group and its lowest lane updates the shared histogram once
            const u32 act = __ballot_sync(0xffffffffu, valid);
            if (valid) {
                const u32 grp = __match_any_sync(act, bin);
                u32 sh = 0, sl = 0;
                if (MODE < 2) { sh = __reduce_add_sync(grp, h); sl = __reduce_add_sync(grp, l); }
                const u32 alo = __reduce_and_sync(grp, (u32)x), ahi = __reduce_and_sync(grp, (u32)(x >> 32));
                const u32 olo = __reduce_or_sync(grp, (u32)x), ohi = __reduce_or_sync(grp, (u32)(x >> 32));
                if (lane == __ffs(grp) - 1) {
                    atomicAdd(&scnt[bin], (u32)__popc(grp));
                    if (MODE < 2) { atomicAdd(&shi[bin], (u64)sh); atomicAdd(&slo[bin], (u64)sl); }
                    atomicAnd(&sand_lo[bin], alo); atomicAnd(&sand_hi[bin], ahi);
                    atomicOr(&sor_lo[bin], olo); atomicOr(&sor_hi[bin], ohi);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < RS_BINS; i += SV_THREADS) {
        const u32 c = scnt[i];
        if (c) {
            atomicAdd(&hist[H_CNT + i], (u64)c);
            if (MODE < 2) { atomicAdd(&hist[H_SHI + i], shi[i]); atomicAdd(&hist[H_SLO + i], slo[i]); }
            atomicAnd(&hist[H_AND + i], ((u64)sand_hi[i] << 32) | sand_lo[i]);
            atomicOr(&hist[H_OR + i], ((u64)sor_hi[i] << 32) | sor_lo[i]);
        }
    }
}

template <int MODE>
static int launch_pass(const double2* amps, const u64* lkeys, u64 n, const SelState* ss, u64* hist, cudaStream_t st) {
    const size_t smem = (size_t)RS_BINS * (5 * 4 + (MODE < 2 ? 16 : 0));
    static bool attr[SV_MAX_DEV];
    sv_set_smem_once(sel_pass_kernel<MODE>, smem, attr);
    u64 blocks = (n + SV_THREADS * SP_IT - 1) / (SV_THREADS * SP_IT);
    const u64 maxb = (u64)sv_sm_count() * (MODE < 2 ? 3 : 4);
    if (blocks > maxb) blocks = maxb;
    if (blocks < 1) blocks = 1;
    sel_pass_kernel<MODE><<<(unsigned)blocks, SV_THREADS, smem, st>>>(amps, lkeys, n, ss, hist);
    return 1;
}
int svk_sel_pass(int mode, const double2* amps, const u64* lkeys, u64 n, const SelState* ss, u64* hist, cudaStream_t st) {
    if (mode == 0) return launch_pass<0>(amps, lkeys, n, ss, hist, st);
    if (mode == 1) return launch_pass<1>(amps, lkeys, n, ss, hist, st);
    return launch_pass<2>(amps, lkeys, n, ss, hist, st);
}

// Tie phase: logical keys of the terms whose probability pattern equals the cutoff PT,
// appended (order irrelevant) to lk_out; their count, AND and OR go to hist[H_EXT..].
__global__ void __launch_bounds__(SV_THREADS) sel_extract_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps,
                                                                 u64 n, const SelState* __restrict__ ssp, KeyMap km,
                                                                 u64* __restrict__ lk_out, u64* __restrict__ hist) {
    if (ssp->done != 0 || ssp->phase != 2) return;
    const u64 PT = ssp->PT;
    const int lane = threadIdx.x & 31;
    u64 a_and = ~0ull, a_or = 0;
    const u64 chunk = (u64)SV_THREADS * SP_IT;
    const u64 nchunks = (n + chunk - 1) / chunk;
    for (u64 c = blockIdx.x; c < nchunks; c += gridDim.x) {
        u64 pat[SP_IT];
#pragma unroll
        for (int r = 0; r < SP_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            pat[r] = ~0ull;
            if (i < n) {
                const double2 a = ld_stream_d2(amps + i);
                if (!(a.x == 0.0 && a.y == 0.0)) pat[r] = (u64)__double_as_longlong(prob_of(a));   // dead entries never tie
            }
        }
#pragma unroll
        for (int r = 0; r < SP_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            const bool hit = (i < n) && pat[r] == PT;
            const u32 grp = __ballot_sync(0xffffffffu, hit);
            if (grp) {
                u64 base = 0;
                if (lane == __ffs(grp) - 1) base = atomicAdd(&hist[H_EXT], (u64)__popc(grp));
                base = __shfl_sync(0xffffffffu, base, __ffs(grp) - 1);
                if (hit) {
                    const u64 lk = logical_key(keys[i], km);
                    lk_out[base + __popc(grp & ((1u << lane) - 1u))] = lk;
                    a_and &= lk; a_or |= lk;
                }
            }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        a_and &= __shfl_xor_sync(0xffffffffu, a_and, d);
        a_or |= __shfl_xor_sync(0xffffffffu, a_or, d);
    }
    if (lane == 0) { atomicAnd(&hist[H_EXT + 1], a_and); atomicOr(&hist[H_EXT + 2], a_or); }
}
int svk_sel_extract(const u64* keys, const double2* amps, u64 n, const SelState* ss, KeyMap km, u64* lk_out, u64* hist,
                    cudaStream_t st) {
    u64 blocks = (n + SV_THREADS * SP_IT - 1) / (SV_THREADS * SP_IT);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    if (blocks < 1) blocks = 1;
    sel_extract_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, ss, km, lk_out, hist);
    return 1;
}

// Seeds the select state for a run over the candidates of the sampled fast path: what lies
// above the band is already kept, S is known exactly.  done = 3 reports a band miss.
__device__ __forceinline__ dd dd_from_fx(const u64* lohi, int Eref) {
    const dd v = dd_add(dd_scale2(dd_from_u64(lohi[1]), 64), dd_from_u64(lohi[0]));
    return dd_scale2(v, Eref - 1075 - 41);
}
__global__ void sel_seed_kernel(SelState* ss, u64* hist, const SampleCtl* ctl, u64 n_orig, u64 max_terms, double min_mass,
                                const PreCut* pre) {
    for (int i = threadIdx.x; i < H_TOTAL; i += blockDim.x)
        hist[i] = ((i >= H_AND && i < H_OR) || i == H_EXT + 1) ? ~0ull : 0ull;
    if (threadIdx.x != 0) return;
    const SampleCtl c = *ctl;
    SelState s;
    memset(&s, 0, sizeof(s));
    s.seeded = 1;
    s.n_total = c.cand_cnt;
    s.cand_count = c.cand_cnt;
    s.below_cnt = c.below_cnt;
    s.P_lo = c.P_lo;
    s.min_mass = min_mass;
    dd tot = dd_from_fx(c.tot, c.Eref);
    const dd abv = dd_from_fx(c.abv, c.Eref);
    if (pre) {   // outputs a fused apply + truncate never wrote: below every stored term, part of S
        dd pm; pm.hi = pre->mass_hi; pm.lo = pre->mass_lo;
        tot = dd_add(tot, pm);
        s.pre_hi = pm.hi; s.pre_lo = pm.lo;
        s.below_cnt += pre->cnt;
    }
    s.total_hi = tot.hi; s.total_lo = tot.lo;
    s.kept_hi = abv.hi; s.kept_lo = abv.lo;
    s.kept_count = c.above_cnt;
    bool miss = c.overflow != 0 || c.cand_cnt == 0 || c.above_cnt + c.below_cnt + c.cand_cnt != n_orig;
    s.count_active = (max_terms != 0 && max_terms < n_orig) ? 1 : 0;
    if (s.count_active) {
        if (max_terms <= c.above_cnt) miss = true; else s.k_rem = max_terms - c.above_cnt;
    }
    s.mass_active = (min_mass < 1.0) ? 1 : 0;
    if (s.mass_active) {
        const dd rem = dd_sub(dd_make(__dmul_rn(min_mass, tot.hi)), abv);
        if (!(rem.hi > 0.0)) miss = true;
        s.mass_rem_hi = rem.hi; s.mass_rem_lo = rem.lo;
    }
    // The candidates lie in [P_lo, P_hi].  When both share the exponent field the exponent level would find one bin:
    // start at the first pattern level instead, with the common leading bits of the band already resolved.
    if (!miss && c.P_hi != ~0ull && (c.P_lo >> 52) == (c.P_hi >> 52) && c.P_lo != c.P_hi) {
        const int e = (int)(c.P_lo >> 52) & 0x7ff;
        const int hb = 63 - __clzll((long long)(c.P_lo ^ c.P_hi));          // highest bit in which the band's ends differ
        const u64 low = (hb >= 63) ? ~0ull : ((2ull << hb) - 1);
        s.E = e ? e : 1;
        s.rmask = ~low; s.rval = c.P_lo & ~low;
        s.dmask = top_bits(low, 11);
        s.phase = 1;
    }
    if (miss) s.done = 3;
    *ss = s;
}
int svk_sel_seed(SelState* ss, u64* hist, const SampleCtl* ctl, u64 n_orig, u64 max_terms, double min_mass, cudaStream_t st,
                 const PreCut* pre) {
    sel_seed_kernel<<<1, SV_THREADS, 0, st>>>(ss, hist, ctl, n_orig, max_terms, min_mass, pre);
    return 1;
}

// ---------------------------------------------------------------------------------------
// one decision step (one block; thread 0 decides), then the histogram is cleared
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ dd prod_u64_double(u64 t, double pv) {   // t * pv, exact to double-double
    const double td = (double)t;                                     // t < 2^53 in practice
    const double hi = __dmul_rn(td, pv);
    return two_sum(hi, __fma_rn(td, pv, -hi));
}

__global__ void __launch_bounds__(SV_THREADS) sel_step_kernel(SelState* ssp, u64* hist, int expected_phase) {
    // expected_phase >= 0: the step of a pass that was launched ahead; it only runs if that pass ran
    if (expected_phase >= 0 && (ssp->done != 0 || ssp->phase != expected_phase)) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* h = reinterpret_cast<u64*>(smem_raw);
    for (int i = threadIdx.x; i < H_TOTAL; i += SV_THREADS) {
        h[i] = hist[i];
        hist[i] = ((i >= H_AND && i < H_OR) || i == H_EXT + 1) ? ~0ull : 0ull;
    }
    __syncthreads();
    SelState s = *ssp;
    const u64* cnt = h + H_CNT;
    const u64* shi = h + H_SHI;
    const u64* slo = h + H_SLO;
    const u64* band = h + H_AND;
    const u64* bor = h + H_OR;
    // per-bin masses and per-segment (8 bins per thread) sums, in parallel; the cut is then found by
    // one thread that skips whole segments and walks only the segment(s) a cut can fall in
    double* mh = reinterpret_cast<double*>(h + H_TOTAL);
    double* ml = mh + RS_BINS;
    double* sgh = ml + RS_BINS;
    double* sgl = sgh + SV_THREADS;
    u64* sgc = reinterpret_cast<u64*>(sgl + SV_THREADS);
    constexpr int SEG = RS_BINS / SV_THREADS;
    const bool l0 = s.phase == 0;
#define BIN_E(d) (l0 ? ((((d) & 0x7ff) != 0) ? ((d) & 0x7ff) : 1) : s.E)
    if (s.phase <= 1) {
        dd sm = dd_make(0.0); u64 sc = 0;
        for (int d = threadIdx.x * SEG + SEG - 1; d >= (int)threadIdx.x * SEG; --d) {
            dd m = dd_make(0.0);
            if (cnt[d]) { m = bin_mass(shi[d], slo[d], BIN_E(d)); sm = dd_add(sm, m); sc += cnt[d]; }
            mh[d] = m.hi; ml[d] = m.lo;
        }
        sgh[threadIdx.x] = sm.hi; sgl[threadIdx.x] = sm.lo; sgc[threadIdx.x] = sc;
    }
    __syncthreads();
    if (threadIdx.x >= 32) return;
    const int lane = threadIdx.x;
    if (s.phase > 1 && lane != 0) return;
    dd kept; kept.hi = s.kept_hi; kept.lo = s.kept_lo;
    dd rem; rem.hi = s.mass_rem_hi; rem.lo = s.mass_rem_lo;
    if (s.phase <= 1) {
        // The cut is found by warp 0: lane L owns segments 8L .. 8L+7 (64 bins).  A suffix scan over the lanes gives
        // every lane the count and the mass ABOVE its bins; each lane then walks its own bins, highest first, and the
        // highest lane that meets a criterion holds its cut bin (counts and masses only grow downwards).
        constexpr int LSEG = SV_THREADS / 32;
        dd lsum = dd_make(0.0); u64 lcnt = 0;
        for (int t = lane * LSEG + LSEG - 1; t >= lane * LSEG; --t)
            if (sgc[t]) { dd x; x.hi = sgh[t]; x.lo = sgl[t]; lsum = dd_add(lsum, x); lcnt += sgc[t]; }
        dd inc = lsum; u64 cinc = lcnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            dd o; o.hi = __shfl_down_sync(0xffffffffu, inc.hi, d); o.lo = __shfl_down_sync(0xffffffffu, inc.lo, d);
            const u64 oc = __shfl_down_sync(0xffffffffu, cinc, d);
            if (lane + d < 32) { inc = dd_add(inc, o); cinc += oc; }
        }
        dd cum; cum.hi = __shfl_down_sync(0xffffffffu, inc.hi, 1); cum.lo = __shfl_down_sync(0xffffffffu, inc.lo, 1);
        u64 cumc = __shfl_down_sync(0xffffffffu, cinc, 1);
        if (lane == 31) { cum = dd_make(0.0); cumc = 0; }
        dd all; all.hi = __shfl_sync(0xffffffffu, inc.hi, 0); all.lo = __shfl_sync(0xffffffffu, inc.lo, 0);   // all candidates
        const u64 allc = __shfl_sync(0xffffffffu, cinc, 0);
        if (l0 && !s.seeded) {   // total mass S and the p-mass threshold min_mass * S (reading R5)
            dd tot = all;
            { dd pm; pm.hi = s.pre_hi; pm.lo = s.pre_lo; tot = dd_add(tot, pm); }
            s.total_hi = tot.hi; s.total_lo = tot.lo;
            rem = dd_make(__dmul_rn(s.min_mass, tot.hi));
        }
        int dK = -1, dM = -1, dlow = -1;
        u64 aboveC_K = 0, aboveC_M = 0; dd aboveM_K = dd_make(0.0), aboveM_M = dd_make(0.0);
        for (int d = (lane * LSEG + LSEG) * SEG - 1; d >= lane * LSEG * SEG; --d) {
            const u64 c = cnt[d];
            if (!c) continue;
            dlow = d;
            dd m; m.hi = mh[d]; m.lo = ml[d];
            if (s.count_active && dK < 0 && cumc + c >= s.k_rem) { dK = d; aboveC_K = cumc; aboveM_K = cum; }
            if (s.mass_active && dM < 0 && dd_ge(dd_add(cum, m), rem)) { dM = d; aboveC_M = cumc; aboveM_M = cum; }
            cumc += c; cum = dd_add(cum, m);
        }
        {   // the highest lane that found a cut bin holds the first crossing; the lowest lane with a bin holds dlow
            const u32 bK = __ballot_sync(0xffffffffu, dK >= 0), bM = __ballot_sync(0xffffffffu, dM >= 0);
            const u32 bL = __ballot_sync(0xffffffffu, dlow >= 0);
            const int lK = bK ? 31 - __clz(bK) : 0, lM = bM ? 31 - __clz(bM) : 0, lL = bL ? __ffs(bL) - 1 : 0;
            dK = __shfl_sync(0xffffffffu, dK, lK); aboveC_K = __shfl_sync(0xffffffffu, aboveC_K, lK);
            aboveM_K.hi = __shfl_sync(0xffffffffu, aboveM_K.hi, lK); aboveM_K.lo = __shfl_sync(0xffffffffu, aboveM_K.lo, lK);
            dM = __shfl_sync(0xffffffffu, dM, lM); aboveC_M = __shfl_sync(0xffffffffu, aboveC_M, lM);
            aboveM_M.hi = __shfl_sync(0xffffffffu, aboveM_M.hi, lM); aboveM_M.lo = __shfl_sync(0xffffffffu, aboveM_M.lo, lM);
            dlow = __shfl_sync(0xffffffffu, dlow, lL);
            if (!bK) dK = -1;
            if (!bM) dM = -1;
            if (!bL) dlow = -1;
        }
        if (lane != 0) return;
        cumc = allc; cum = all;     // totals over the candidates, as the sequential walk would leave them
        if (dlow < 0) { s.done = s.seeded ? 3 : 1; s.PT = 0; s.KT = ~0ull; }   // no candidates at all
        else if (s.seeded && s.below_cnt > 0 && (!s.mass_active || dM < 0) && (!s.count_active || dK < 0)) {
            s.done = 3;             // the cut lies below the sampled band: the caller runs the full select
        } else {
            // threshold not reached (rounding of min_mass * S): every candidate is needed
            if (s.mass_active && dM < 0) {
                dM = dlow; aboveC_M = cumc - cnt[dlow];
                aboveM_M = dd_sub(cum, bin_mass(shi[dlow], slo[dlow], BIN_E(dlow))); rem = cum;
            }
            if (s.count_active && dK < 0) {
                dK = dlow; aboveC_K = cumc - cnt[dlow];
                aboveM_K = dd_sub(cum, bin_mass(shi[dlow], slo[dlow], BIN_E(dlow))); s.k_rem = cumc;
            }
            if (s.count_active && s.mass_active) {
                if (dK > dM) s.mass_active = 0; else if (dM > dK) s.count_active = 0;
            }
            int dcut; u64 aboveC; dd aboveM;
            if (s.count_active) { dcut = dK; aboveC = aboveC_K; aboveM = aboveM_K; }
            else { dcut = dM; aboveC = aboveC_M; aboveM = aboveM_M; }
            s.kept_count += aboveC; kept = dd_add(kept, aboveM);
            if (s.count_active) s.k_rem -= aboveC;
            if (s.mass_active) rem = dd_sub(rem, aboveM);
            s.cand_count = cnt[dcut];
            const dd bm = bin_mass(shi[dcut], slo[dcut], BIN_E(dcut));
            if (l0) { s.rmask = 0xfffull << 52; s.rval = (u64)dcut << 52; s.E = BIN_E(dcut); }
            else { s.rmask |= s.dmask; s.rval |= pdep_desc((u32)dcut, s.dmask); }
            const u64 A = band[dcut], O = bor[dcut];
            const u64 diff = A ^ O;
            s.rmask |= ~diff; s.rval = A & s.rmask;      // bits common to every candidate are resolved
            bool take_all = false;
            if (s.cand_count == 1) take_all = true;
            else {
                const bool allK = !s.count_active || s.k_rem >= s.cand_count;
                if (!s.mass_active && allK) take_all = true;
                else if (s.mass_active && allK) s.count_active = 0;
            }
            if (take_all) {
                // A <= every member of the bin, > every term in a lower bin; seeded: the terms below
                // the band never entered the histograms, P_lo separates them from every candidate
                s.PT = (s.seeded && A < s.P_lo) ? s.P_lo : A; s.KT = ~0ull;
                s.kept_count += s.cand_count; kept = dd_add(kept, bm);
                s.done = 1;
            } else if (diff == 0) {                      // the candidates are exact ties at probability pv
                const double pv = __longlong_as_double((long long)A);
                u64 t = s.cand_count;
                if (s.count_active && s.k_rem < t) t = s.k_rem;
                if (s.mass_active) {                     // smallest tm with tm * pv >= rem
                    const double qd = ceil(rem.hi / pv);
                    u64 tm = !(qd >= 1.0) ? 1 : (qd > 9.0e18 ? s.cand_count : (u64)qd);
                    if (tm > s.cand_count) tm = s.cand_count;
                    while (tm > 1 && dd_ge(prod_u64_double(tm - 1, pv), rem)) --tm;
                    while (tm < s.cand_count && !dd_ge(prod_u64_double(tm, pv), rem)) ++tm;
                    if (tm < t) t = tm;
                }
                if (t < 1) t = 1;
                s.PT = A;
                kept = dd_add(kept, prod_u64_double(t, pv));   // t tied terms are kept in any case
                if (t >= s.cand_count) { s.KT = ~0ull; s.kept_count += s.cand_count; s.done = 1; }
                else { s.k_rem = t; s.tie_total = s.cand_count; s.count_active = 1; s.mass_active = 0; s.phase = 2; }
            } else {
                s.dmask = top_bits(diff, 11);
                s.phase = 1;
            }
        }
#undef BIN_E
    } else if (s.phase == 2) {      // the tied keys have been extracted
        const u64 got = h[H_EXT], A = h[H_EXT + 1], O = h[H_EXT + 2];
        if (got != s.tie_total) { s.done = 2; }   // internal inconsistency, reported by the host
        else {
            const u64 diff = A ^ O;
            s.krmask = 0; s.krval = 0;
            s.kdmask = top_bits(diff, 11);
            s.phase = 3;
        }
    } else {                        // key level: lower logical keys are kept first (reading R4)
        u64 cumc = 0; int dcut = -1;
        for (int d = 0; d < RS_BINS; ++d) {
            if (!cnt[d]) continue;
            dcut = d;
            if (cumc + cnt[d] >= s.k_rem) break;
            cumc += cnt[d];
        }
        if (dcut < 0) { s.done = 2; }
        else {
            s.kept_count += cumc; s.k_rem -= cumc;
            s.krmask |= s.kdmask; s.krval |= pdep_desc((u32)dcut, s.kdmask);
            s.cand_count = cnt[dcut];
            const u64 A = band[dcut], O = bor[dcut];
            if (s.k_rem >= s.cand_count) {       // the whole bin is kept: O >= its members, < every higher bin
                s.KT = O; s.kept_count += s.cand_count; s.done = 1;
            } else {
                const u64 diff = A ^ O;
                s.krmask |= ~diff; s.krval = A & s.krmask;
                s.kdmask = top_bits(diff, 11);
                if (diff == 0) s.done = 2;       // duplicate keys: cannot happen
            }
        }
    }
    s.kept_hi = kept.hi; s.kept_lo = kept.lo;
    s.mass_rem_hi = rem.hi; s.mass_rem_lo = rem.lo;
    if (s.done == 1) {
        s.kept_mass = kept.hi; s.total_mass = s.total_hi;
        s.scale = __ddiv_rn(1.0, __dsqrt_rn(s.kept_mass));
        s.kept_fraction = __ddiv_rn(s.kept_mass, s.total_mass);
        s.final_count = s.kept_count;
    }
    *ssp = s;
}
int svk_sel_step(SelState* ss, u64* hist, cudaStream_t st, int expected_phase) {
    const size_t smem = (size_t)H_TOTAL * 8 + (size_t)RS_BINS * 16 + (size_t)SV_THREADS * 24;
    static bool attr[SV_MAX_DEV];
    sv_set_smem_once(sel_step_kernel, smem, attr);
    sel_step_kernel<<<1, SV_THREADS, smem, st>>>(ss, hist, expected_phase);
    return 1;
}

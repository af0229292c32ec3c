// Truncation cut, fast path.
//
// The paper sorts all terms by probability; sv_radix_select.cu finds the cut with several
// histogram passes over the whole state.  Here ONE streaming pass over the amplitudes is
// enough in the common case:
//
//   1. sample     M evenly spaced terms -> the top 24 bits of their probability patterns,
//                 sorted (a 0.5 MB LSD radix sort that lives in L2);
//   2. pivots     from the sorted sample, two patterns P_lo <= P_hi that bracket the cut
//                 with wide statistical margins, for the top-k criterion (a quantile) and
//                 for the p-mass criterion (the tail of the sample whose scaled mass is
//                 the mass to be dropped);
//   3. classify   one pass: every term is "above" (pattern > P_hi: certainly kept), "below"
//                 (pattern < P_lo: certainly dropped) or a candidate.  The pass returns the
//                 EXACT count and mass above, the exact total mass S, the count below, and
//                 copies the candidates (a few per cent of the state) to the idle buffers;
//   4. finish     the exact adaptive radix select of sv_radix_select.cu runs on the
//                 candidates only, seeded with what is already kept.
//
// The pivots only steer the work.  The cut itself is exact: if it turns out not to lie
// among the candidates (or a probability is out of the fixed-point range) the seeded select
// reports a band miss and the caller falls back to the full-state select.
//
// Exact masses (D3): p is converted to a 128-bit fixed-point integer relative to
// a reference exponent, and integers are added -- the sums do not depend on the order in
// which threads or blocks add them.
#include "sv_tile.cuh"
#include "sv_launch.cuh"

typedef unsigned __int128 u128;

// The sample keeps the top 24 bits of a probability pattern (sign, exponent, 12 mantissa bits: 2.4e-4
// relative resolution, far finer than the statistical margins of the pivots): three 8-bit sort passes.
#define SS_DROP 40

// XF (fused diagonal gate + truncate, sv_apply_gate_truncate): the diagonal gate that precedes the truncation
// has NOT been applied yet.  The sample and the classification pass see every amplitude as that gate leaves
// it -- pending cut (dropped -> dead entry 0+0i), renormalisation, phase, exactly the arithmetic of
// diag_kernel / diag_pend_kernel -- and the classification pass writes it back in place: the gate and the
// truncation's pass over the state are ONE pass (key read, amplitude read + write: 40 B per term).
__device__ __forceinline__ double2 xf_amp(double2 a, u64 k, const PendPred& pd, const double2* sd, const int* cpos, int mc) {
    if (pd.active) {
        if (a.x == 0.0 && a.y == 0.0) return a;                       // dead stays dead
        if (!pend_keep(pd, k, a)) return make_double2(0.0, 0.0);
        a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale);
    }
    int cx = 0;
    for (int j = 0; j < mc; ++j) cx |= (int)((k >> cpos[j]) & 1ull) << j;
    const double2 u = sd[cx];
    double2 o;
    o.x = __dsub_rn(__dmul_rn(u.x, a.x), __dmul_rn(u.y, a.y));
    o.y = __dadd_rn(__dmul_rn(u.x, a.y), __dmul_rn(u.y, a.x));
    return o;
}

template <bool XF>
__global__ void __launch_bounds__(SV_THREADS) ss_sample_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps, u64 n, u32 M,
                                                               u64* __restrict__ smp, PendPred pd, const GateTab* __restrict__ gtab) {
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    const u64 i = (u64)(((u128)j * n) / M);
    double2 a = ld_stream_d2(amps + i);
    if (XF) a = xf_amp(a, keys[i], pd, gtab->U, gtab->ctrl_pos, gtab->mc);
    // dead entries (0+0i) sort to the front as key 0; live terms get their pattern's top 24 bits + 1
    smp[j] = (a.x == 0.0 && a.y == 0.0) ? 0ull : (((u64)__double_as_longlong(prob_of(a)) >> SS_DROP) + 1ull);
}

__device__ __forceinline__ double smp_prob(u64 top) {   // mid-point of the values sharing these top bits
    return __longlong_as_double((long long)((top << SS_DROP) | (1ull << (SS_DROP - 1))));
}

// One block of 1024 threads.  smp[0..M) ascending; the first z entries are 0 (dead sample points),
// the live ones hold (top 32 pattern bits) + 1.  Warp w owns a contiguous range of the live part
// and walks it 32 elements at a time.
__global__ void __launch_bounds__(1024) ss_pivot_kernel(const u64* __restrict__ smp, u32 M, u64 n_live, u64 max_terms,
                                                        double min_mass, double mass_est, SampleCtl* __restrict__ ctl,
                                                        const PreCut* __restrict__ precut) {
    __shared__ double wsum[32];
    __shared__ u32 cnt[2][3];   // [sweep][threshold]
    __shared__ u32 s_z;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {   // z = number of dead sample points (lower bound of 1)
        u32 lo = 0, hi = M;
        while (lo < hi) { const u32 mid = (lo + hi) >> 1; if (smp[mid] == 0) lo = mid + 1; else hi = mid; }
        s_z = lo;
    }
    if (threadIdx.x < 6) cnt[threadIdx.x / 3][threadIdx.x % 3] = 0;
    __syncthreads();
    const u32 z = s_z, Ml = M - z;
    const u64* live = smp + z;
    const u32 per = (Ml + 31) / 32;
    const u32 b0 = min(Ml, warp * per), b1 = min(Ml, b0 + per);
    double s = 0.0;
#pragma unroll 8
    for (u32 i = b0 + lane; i < b1; i += 32) s += smp_prob(live[i] - 1);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (lane == 0) wsum[warp] = s;
    __syncthreads();
    double pre = 0.0, T = 0.0;
    for (int w = 0; w < 32; ++w) { if (w < warp) pre += wsum[w]; T += wsum[w]; }
    const bool mass_on = min_mass < 1.0 && Ml > 0;
    // mass to drop, in sample units (the tail is made of small terms, so the scaled sample tail
    // estimates it well even when a few heavy terms carry most of S)
    const double per_sample = (double)n_live / (double)max(Ml, 1u);
    // a fused apply + truncate has left D_pre of the mass out already (all of it below every stored term)
    const double D_pre = precut ? precut->mass_hi : 0.0;
    const double S_est = (mass_est == mass_est && mass_est > 0.0) ? mass_est : T * per_sample + D_pre;
    const double X0 = fmax(0.0, (1.0 - min_mass) * S_est - D_pre) / per_sample;
    // sweep 1: a0 = sample elements in the nominal tail; sweep 2: the band X0 / (1 + eps) .. X0 * (1 + eps)
    // with eps ~ 10 / sqrt(a0) (the relative noise of a tail sum of a0 sampled terms)
    double X[3] = {X0, X0, X0};
    for (int sweep = 0; sweep < 2 && mass_on; ++sweep) {
        u32 c[3] = {0, 0, 0};
        double run = pre;
        for (u32 ib = b0; ib < b1; ib += 32 * 8) {   // 8 rows of 32 per batch: the loads of a batch are in flight together
            double vv[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const u32 i = ib + u * 32 + lane;
                vv[u] = (i < b1) ? smp_prob(live[i] - 1) : 0.0;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const u32 i = ib + u * 32 + lane;
                double inc = vv[u];
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const double t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                const double incl = run + inc;   // mass of the sample's i + 1 smallest live elements
                if (i < b1) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) c[k] += (incl <= X[k]) ? 1u : 0u;
                }
                run += __shfl_sync(0xffffffffu, inc, 31);
            }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            u32 v = c[k];
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            if (lane == 0 && v) atomicAdd(&cnt[sweep][k], v);
        }
        __syncthreads();
        if (sweep == 0) {
            const double a0 = (double)cnt[0][1];
            const double eps = fmin(2.0, 10.0 / sqrt(fmax(a0, 1.0)));
            X[0] = X0 / (1.0 + eps); X[2] = X0 * (1.0 + eps);
        }
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    // numbers of (smallest) live sample elements certainly / possibly dropped
    long long lo_idx = 0, hi_idx = 0;
    if (mass_on) {
        const long long a0 = cnt[0][1];
        long long a_lo = (a0 < 128) ? 0 : (long long)cnt[1][0] - 8;
        long long a_hi = (a0 < 128) ? max((long long)cnt[1][2] + 8, 2 * a0 + 64) : (long long)cnt[1][2] + 8;
        lo_idx = max(lo_idx, a_lo); hi_idx = max(hi_idx, a_hi);
    }
    if (max_terms != 0 && max_terms < n_live) {
        const double q = (double)(n_live - max_terms) / (double)n_live;
        const double d = q * (double)Ml;
        const double dl = 6.0 * sqrt(fmax(d * (1.0 - q), 0.0)) + 8.0;
        lo_idx = max(lo_idx, (long long)floor(d - dl));
        hi_idx = max(hi_idx, (long long)ceil(d + dl));
    }
    SampleCtl c;
    memset(&c, 0, sizeof(c));
    c.P_lo = (lo_idx <= 0 || Ml == 0) ? 0ull : ((live[min((long long)Ml, lo_idx) - 1] - 1) << SS_DROP);
    c.P_hi = (hi_idx >= (long long)Ml) ? ~0ull : (((live[hi_idx] - 1) << SS_DROP) | ((1ull << SS_DROP) - 1));
    int er = (Ml ? (int)((live[Ml - 1] - 1) >> (52 - SS_DROP)) : 1023) + 12;
    c.Eref = er > 2046 ? 2046 : er;
    *ctl = c;
}

// p (as its bit pattern) in units of 2^(Eref - 1075 - 41); exponents above Eref overflow
__device__ __forceinline__ u128 fx_of(u64 pat, int Eref, u32& ovf) {
    int e = (int)(pat >> 52);
    u64 M = pat & ((1ull << 52) - 1);
    if (e) M |= 1ull << 52; else e = 1;
    const int sh = e - Eref + 41;
    if (sh > 41) { ovf = 1; return 0; }
    if (sh >= 0) return (u128)M << sh;
    if (sh > -53) return (u128)(M >> (-sh));
    return 0;
}
__device__ __forceinline__ u128 warp_sum_u128(u128 v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const u64 lo = __shfl_xor_sync(0xffffffffu, (u64)v, d);
        const u64 hi = __shfl_xor_sync(0xffffffffu, (u64)(v >> 64), d);
        v += ((u128)hi << 64) | lo;
    }
    return v;
}
__device__ __forceinline__ void atomic_add_u128(u64* lohi, u128 v) {   // lohi[0] = low word, lohi[1] = high word
    const u64 lo = (u64)v, hi = (u64)(v >> 64);
    const u64 old = atomicAdd(&lohi[0], lo);
    const u64 carry = (old + lo < old) ? 1ull : 0ull;
    if (hi + carry) atomicAdd(&lohi[1], hi + carry);
}

#define SC_IT 4
#define SC_WBUF 96       // candidate slots per warp (flushed when more than 64 are waiting)
// Candidates are rare (a few per cent) but almost every warp meets one every few iterations.  They
// are parked in a warp-private shared-memory buffer (amplitude + index) and flushed 64+ at a
// time: one global atomic and one batch of key loads per flush instead of one per iteration.
template <bool XF>
__global__ void __launch_bounds__(SV_THREADS) ss_classify_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps,
                                                                 u64 n, SampleCtl* __restrict__ ctl, u64* __restrict__ ckeys,
                                                                 double2* __restrict__ camps, unsigned char* __restrict__ seg_cnt,
                                                                 double2* amps_rw, PendPred pd, const GateTab* __restrict__ gtab) {
    __shared__ double2 s_ba[SV_THREADS / 32][SC_WBUF];
    __shared__ u64 s_bi[SV_THREADS / 32][SC_WBUF];
    __shared__ double2 sd[16];
    __shared__ int s_cpos[SV_MAX_M], s_mc;
    if (XF) {
        if (threadIdx.x < 16) sd[threadIdx.x] = gtab->U[threadIdx.x];
        if (threadIdx.x < SV_MAX_M) s_cpos[threadIdx.x] = gtab->ctrl_pos[threadIdx.x];
        if (threadIdx.x == 0) s_mc = gtab->mc;
        __syncthreads();
    }
    const int mc = XF ? s_mc : 0;
    const u64 P_hi = ctl->P_hi, P_lo = ctl->P_lo;
    const int Eref = ctl->Eref;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double2* ba = s_ba[warp];
    u64* bi = s_bi[warp];
    int nbuf = 0;            // warp-uniform
    auto flush = [&]() {
        u64 base = 0;
        if (lane == 0) base = atomicAdd(&ctl->cand_cnt, (u64)nbuf);
        base = __shfl_sync(0xffffffffu, base, 0);
        for (int q = lane; q < nbuf; q += 32) {
            ckeys[base + q] = keys[bi[q]];
            camps[base + q] = ba[q];
        }
        __syncwarp();
        nbuf = 0;
    };
    u128 tot = 0, abv = 0;
    u32 n_abv = 0, n_blw = 0, ovf = 0;
    const u64 chunk = (u64)SV_THREADS * SC_IT;
    const u64 nchunks = (n + chunk - 1) / chunk;
    for (u64 c = blockIdx.x; c < nchunks; c += gridDim.x) {
        double2 a[SC_IT];
        u64 kx[XF ? SC_IT : 1];
#pragma unroll
        for (int r = 0; r < SC_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            if (XF) {
                a[r] = (i < n) ? amps_rw[i] : make_double2(0.0, 0.0);
                kx[r] = (i < n) ? ld_stream_u64(keys + i) : 0ull;
            } else {
                a[r] = (i < n) ? ld_stream_d2(amps + i) : make_double2(0.0, 0.0);
            }
        }
        if (XF) {
#pragma unroll
            for (int r = 0; r < SC_IT; ++r) {
                const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
                if (i < n && !(pd.active && a[r].x == 0.0 && a[r].y == 0.0)) {   // (a dead entry is not rewritten)
                    a[r] = xf_amp(a[r], kx[r], pd, sd, s_cpos, mc);
                    amps_rw[i] = a[r];
                }
            }
        }
#pragma unroll
        for (int r = 0; r < SC_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            const bool ok = i < n && !(a[r].x == 0.0 && a[r].y == 0.0);   // dead entries take no part
            const u64 pat = (u64)__double_as_longlong(prob_of(a[r]));
            const u128 f = ok ? fx_of(pat, Eref, ovf) : (u128)0;
            tot += f;
            const bool above = ok && pat > P_hi, below = ok && pat < P_lo;
            if (above) { abv += f; ++n_abv; }
            n_blw += below ? 1u : 0u;
            const bool cand = ok && !above && !below;
            const u32 grp = __ballot_sync(0xffffffffu, cand);
            if (seg_cnt) {   // entries of this 32-entry segment that a band compaction would keep (above or candidate)
                const u32 nb = __ballot_sync(0xffffffffu, ok && !below);
                if (lane == 0 && (c * chunk + (u64)r * SV_THREADS + (threadIdx.x & ~31)) < n) seg_cnt[(c * chunk + (u64)r * SV_THREADS + threadIdx.x) >> 5] = (unsigned char)__popc(nb);
            }
            if (grp) {
                if (cand) {
                    const int q = nbuf + __popc(grp & ((1u << lane) - 1u));
                    ba[q] = a[r]; bi[q] = i;
                }
                nbuf += __popc(grp);
                __syncwarp();
                if (nbuf > SC_WBUF - 32) flush();
            }
        }
    }
    if (nbuf) flush();
    tot = warp_sum_u128(tot);
    abv = warp_sum_u128(abv);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_abv += __shfl_xor_sync(0xffffffffu, n_abv, d);
        n_blw += __shfl_xor_sync(0xffffffffu, n_blw, d);
        ovf |= __shfl_xor_sync(0xffffffffu, ovf, d);
    }
    if (lane == 0) {
        atomic_add_u128(ctl->tot, tot);
        atomic_add_u128(ctl->abv, abv);
        if (n_abv) atomicAdd(&ctl->above_cnt, (u64)n_abv);
        if (n_blw) atomicAdd(&ctl->below_cnt, (u64)n_blw);
        if (ovf) atomicOr(&ctl->overflow, 1ull);
    }
}

int svk_ss_sample(const double2* amps, u64 n, u32 M, u64* smp, cudaStream_t st, const u64* keys, const PendPred* pd, const GateTab* xf_tab) {
    if (xf_tab) ss_sample_kernel<true><<<(M + SV_THREADS - 1) / SV_THREADS, SV_THREADS, 0, st>>>(keys, amps, n, M, smp, *pd, xf_tab);
    else ss_sample_kernel<false><<<(M + SV_THREADS - 1) / SV_THREADS, SV_THREADS, 0, st>>>(nullptr, amps, n, M, smp, PendPred{}, nullptr);
    return 1;
}
int svk_ss_pivot(const u64* smp_sorted, u32 M, u64 n_live, u64 max_terms, double min_mass, double mass_est, SampleCtl* ctl,
                 cudaStream_t st, const PreCut* pre) {
    ss_pivot_kernel<<<1, 1024, 0, st>>>(smp_sorted, M, n_live, max_terms, min_mass, mass_est, ctl, pre);
    return 1;
}
template <bool XF>
static void launch_classify(const u64* keys, const double2* amps, u64 n, SampleCtl* ctl, u64* ckeys, double2* camps, unsigned char* seg_cnt,
                            cudaStream_t st, double2* amps_rw, const PendPred& pd, const GateTab* tab) {
    static int per_sm_c[SV_MAX_DEV];   // one wave of resident blocks: a grid-stride loop has no tail
    const int per_sm = sv_blocks_per_sm(ss_classify_kernel<XF>, 0, per_sm_c);
    u64 blocks = (n + SV_THREADS * SC_IT - 1) / (SV_THREADS * SC_IT);
    if (blocks > (u64)sv_sm_count() * per_sm) blocks = (u64)sv_sm_count() * per_sm;
    if (blocks < 1) blocks = 1;
    ss_classify_kernel<XF><<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, ctl, ckeys, camps, seg_cnt, amps_rw, pd, tab);
}
int svk_ss_classify(const u64* keys, const double2* amps, u64 n, SampleCtl* ctl, u64* ckeys, double2* camps, unsigned char* seg_cnt,
                    cudaStream_t st, double2* amps_rw, const PendPred* pd, const GateTab* xf_tab) {
    if (xf_tab) launch_classify<true>(keys, amps, n, ctl, ckeys, camps, seg_cnt, st, amps_rw, *pd, xf_tab);
    else launch_classify<false>(keys, amps, n, ctl, ckeys, camps, seg_cnt, st, nullptr, PendPred{}, nullptr);
    return 1;
}

// ---------------------------------------------------------------------------------------
// Band compaction: after a cut that drops a large part of the state (the cap after an expanding gate)
// the entries BELOW the sampled band are squeezed out at once.  The classify pass has left, per
// 32-entry segment, the number of entries that stay (above or candidate); a 1024-entry chunk sums
// its 32 segments, an exclusive scan over the chunk sums gives every chunk its output offset, and
// the scatter pass below needs neither a scan of its own nor a look-back: it streams like the
// classify pass.  Rejected candidates stay behind as (few) dead entries for the pending cut.
// ---------------------------------------------------------------------------------------
__global__ void ss_chunk_sum_kernel(const unsigned char* __restrict__ seg_cnt, u64 nseg, u32 nchunks, u32* __restrict__ chunk_cnt) {
    const u32 c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nchunks) return;
    u32 sum = 0;
    for (int q = 0; q < 32; ++q) { const u64 sidx = (u64)c * 32 + q; if (sidx < nseg) sum += seg_cnt[sidx]; }
    chunk_cnt[c] = sum;
}
__global__ void __launch_bounds__(SV_THREADS) ss_band_compact_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps, u64 n,
                                                                    const SampleCtl* __restrict__ ctl,
                                                                    const unsigned char* __restrict__ seg_cnt, const u32* __restrict__ chunk_off,
                                                                    u64* __restrict__ kout, double2* __restrict__ aout) {
    const u64 P_lo = ctl->P_lo;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const u64 chunk = (u64)SV_THREADS * SC_IT;
    const u64 nchunks = (n + chunk - 1) / chunk;
    const u64 nseg = (n + 31) >> 5;
    for (u64 c = blockIdx.x; c < nchunks; c += gridDim.x) {
        double2 a[SC_IT];
#pragma unroll
        for (int r = 0; r < SC_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            a[r] = (i < n) ? ld_stream_d2(amps + i) : make_double2(0.0, 0.0);
        }
        const u64 sidx = c * 32 + lane;                       // lane l holds segment l of the chunk
        const u32 sc = (sidx < nseg) ? seg_cnt[sidx] : 0u;
        u32 inc = sc;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const u32 t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
        const u32 segoff = inc - sc;
        const u64 cbase = chunk_off[c];
#pragma unroll
        for (int r = 0; r < SC_IT; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            const bool alive = i < n && !(a[r].x == 0.0 && a[r].y == 0.0);
            const bool keep = alive && (u64)__double_as_longlong(prob_of(a[r])) >= P_lo;
            const u32 bal = __ballot_sync(0xffffffffu, keep);
            const u32 off = __shfl_sync(0xffffffffu, segoff, r * (SV_THREADS / 32) + warp);
            if (keep) {
                const u64 pos = cbase + off + __popc(bal & ((1u << lane) - 1u));
                st_stream_u64(kout + pos, ld_stream_u64(keys + i));
                st_stream_d2(aout + pos, a[r]);
            }
        }
    }
}
int svk_ss_band_compact(const u64* keys, const double2* amps, u64 n, const SampleCtl* ctl, const unsigned char* seg_cnt,
                        u32* chunk_cnt, u64* scan_status, u32* tile_counter, u64* kout, double2* aout, cudaStream_t st) {
    const u64 chunk = (u64)SV_THREADS * SC_IT;
    const u32 nchunks = (u32)((n + chunk - 1) / chunk);
    ss_chunk_sum_kernel<<<(nchunks + 255) / 256, 256, 0, st>>>(seg_cnt, (n + 31) >> 5, nchunks, chunk_cnt);
    int launches = 1 + svk_scan_u32(chunk_cnt, nchunks, scan_status, tile_counter, st);
    static int per_sm_c[SV_MAX_DEV];
    const int per_sm = sv_blocks_per_sm(ss_band_compact_kernel, 0, per_sm_c);
    u64 blocks = nchunks;
    if (blocks > (u64)sv_sm_count() * per_sm) blocks = (u64)sv_sm_count() * per_sm;
    ss_band_compact_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, ctl, seg_cnt, chunk_cnt, kout, aout);
    return launches + 1;
}

// Fused apply + truncate ("apply, then truncate"): the cap cut
// is estimated BEFORE the gate's outputs exist, so that the pass never writes what the
// truncation that follows is certain to drop.
//
//   1. pre-sample   M evenly spaced stored entries; each stands for its tuple (the entry and its
//                   partners in the gate's active qubits).  A trial is accepted for
//                   one member per tuple only and emits ONE of the tuple's 2^ma outputs, so every
//                   (tuple, row) pair -- every output the gate can produce -- is drawn with the
//                   same probability 1 / (2^ma n).  The trial computes that output amplitude with
//                   the arithmetic of the pass itself and keeps the top 24 bits of its
//                   probability pattern (0: no output);
//   2. sort         the 0.5 MB LSD radix sort of the truncation's sample (sv_sort.cu);
//   3. pre-pivot    P_floor = the pattern below which, with a 6 sigma margin, at least
//                   max_terms outputs remain.  Outputs with a pattern < P_floor are dropped
//                   by the pass (sv_pair.cu, PRE); their number and mass are carried to the
//                   exact select of the truncation that follows, which sees them as terms below
//                   its band.
//
// The floor only steers: the pass reports how many outputs stayed, and if that is not more than
// max_terms (the margin failed) the caller re-runs the pass without a floor -- its input is intact.
#include "sv_tile.cuh"

#define PS_DROP 40   // as SS_DROP in sv_sample_select.cu: sign, exponent and 12 mantissa bits survive

// Trial t looks at a pseudo-random entry of the t-th of M equal strata and draws a pseudo-random row: evenly spaced
// positions would be correlated with the local index of a term inside its tuple when tuples are stored densely
// (every second entry is a "bit 0" member), which biases the acceptance.  A fixed hash: the same trials every run.
__device__ __forceinline__ u32 ps_hash(u32 x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}
__device__ __forceinline__ u64 ps_position(u32 t, u64 n, u32 M) {
    const unsigned __int128 num = (unsigned __int128)t * n + (((unsigned __int128)ps_hash(t) * n) >> 32);
    const u64 i = (u64)(num / M);
    return i < n ? i : n - 1;
}

__global__ void __launch_bounds__(SV_THREADS) pre_sample1_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps,
                                                                 u64 n, int p, const GateTab* __restrict__ gtab, PendPred pd,
                                                                 u32 M, u64* __restrict__ smp) {
    const u32 t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= M) return;
    const u64 i = ps_position(t, n, M);
    const u64 bit = 1ull << p;
    const u64 himask = (p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    auto live_amp = [&](u64 idx, u64 key) {
        double2 a = amps[idx];
        if (pd.active) {
            if (pend_keep(pd, key, a)) { a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale); }
            else { a.x = 0.0; a.y = 0.0; }
        }
        return a;
    };
    u64 out = 0;
    const u64 k = keys[i];
    const double2 a = live_amp(i, k);
    if (!(a.x == 0.0 && a.y == 0.0)) {
        const int c = (int)((k >> p) & 1ull);
        // the partner (the stored key with bit p flipped), by binary search in the ascending keys
        const u64 kp = k ^ bit;
        u64 lo = c ? 0 : i + 1, hi = c ? i : n;
        while (lo < hi) { const u64 mid = (lo + hi) >> 1; if (keys[mid] < kp) lo = mid + 1; else hi = mid; }
        double2 pa = make_double2(0.0, 0.0);
        if (lo < n && keys[lo] == kp) pa = live_amp(lo, kp);
        const bool has_partner = !(pa.x == 0.0 && pa.y == 0.0);
        if (!(has_partner && c)) {           // one accepted member per tuple: the bit-0 one when both are present
            const u64 nk = (k & himask) | ((k & lowmask) << 1);   // layout after the move, LSB = 0
            int cx = 0;
            const int mc = gtab->mc;
            for (int q = 0; q < mc; ++q) cx |= (int)((nk >> gtab->ctrl_pos[q]) & 1ull) << q;
            const double2* u = &gtab->U[cx << 2];                 // u[xr * 2 + xc]
            const int r = (int)(ps_hash(t ^ 0x9e3779b9u) & 1u);   // the output row this trial draws
            double sr = 0.0, si = 0.0;
            if (!c) {
                cmul_acc(sr, si, u[2 * r].x, u[2 * r].y, a.x, a.y);
                if (has_partner) cmul_acc(sr, si, u[2 * r + 1].x, u[2 * r + 1].y, pa.x, pa.y);
            } else {
                cmul_acc(sr, si, u[2 * r + 1].x, u[2 * r + 1].y, a.x, a.y);
            }
            if (!(sr == 0.0 && si == 0.0))
                out = ((u64)__double_as_longlong(prob_of(make_double2(sr, si))) >> PS_DROP) + 1ull;
        }
    }
    smp[t] = out;
}

// The same for a gate with ma >= 2 active bits (final pass: sv_group.cu).  The tuple of entry i is
// made of up to 2^ma stored entries: with the last active bit still at position p (it moves in the final pass) they
// sit in two runs, one per value of bit p, each a range of keys that agree above the ma - 1 low bits; without a
// move (p < 0) in one run.  The trial is accepted for the live member with the smallest local index only and draws
// ONE of the 2^ma output rows: every (tuple, row) pair has the probability 1 / (2^ma n).
__global__ void __launch_bounds__(SV_THREADS) pre_sample_group_kernel(const u64* __restrict__ keys, const double2* __restrict__ amps,
                                                                      u64 n, int p, int ma, const GateTab* __restrict__ gtab, PendPred pd,
                                                                      u32 M, u64* __restrict__ smp, int p2) {
    const u32 t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= M) return;
    const u64 i = ps_position(t, n, M);
    const bool mv = p >= 0;
    const bool two = mv && p2 >= 0;        // the final pass moves two bits (p > p2): the members sit in four runs
    const int np = 1 << ma;
    const u64 AM = (u64)np - 1;
    const u64 bit = mv ? (1ull << p) : 0ull;
    const u64 himask = (!mv || p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    const u64 bit2 = two ? (1ull << p2) : 0ull;
    const u64 midmask = two ? ((bit - 1) & ~((bit2 << 1) - 1)) : 0ull, lowmask2 = two ? (bit2 - 1) : 0ull;
    auto new_key = [&](u64 k) {
        if (two) return (k & himask) | ((k & midmask) << 1) | ((k & lowmask2) << 2) | (((k >> p) & 1ull) << 1) | ((k >> p2) & 1ull);
        return mv ? ((k & himask) | ((k & lowmask) << 1) | ((k >> p) & 1ull)) : k;
    };
    auto live_amp = [&](u64 idx, u64 key) {
        double2 a = amps[idx];
        if (pd.active) {
            if (pend_keep(pd, key, a)) { a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale); }
            else { a.x = 0.0; a.y = 0.0; }
        }
        return a;
    };
    u64 out = 0;
    const u64 k = keys[i];
    const double2 a_i = live_amp(i, k);
    if (!(a_i.x == 0.0 && a_i.y == 0.0)) {
        const u64 nk = new_key(k);
        double2 av[16];
        u32 pm = 0;
        // the runs of stored keys that hold the tuple's members
        const u64 low = two ? (((u64)np >> 2) - 1) : (mv ? (((u64)np >> 1) - 1) : AM);   // stored low bits that vary inside a run
        const int nruns = two ? 4 : (mv ? 2 : 1);
        for (int rr = 0; rr < nruns; ++rr) {
            const u64 base = two ? (((k & ~bit & ~bit2) & ~low) | ((rr & 2) ? bit : 0ull) | ((rr & 1) ? bit2 : 0ull))
                                 : (mv ? (((k & ~bit) & ~low) | (rr ? bit : 0ull)) : (k & ~low));
            u64 lo = 0, hi = n;
            while (lo < hi) { const u64 mid = (lo + hi) >> 1; if (keys[mid] < base) lo = mid + 1; else hi = mid; }
            for (u64 j = lo; j < n && j <= lo + low; ++j) {
                const u64 kj = keys[j];
                if ((kj & ~low) != base) break;
                const double2 aj = (j == i) ? a_i : live_amp(j, kj);
                if (!(aj.x == 0.0 && aj.y == 0.0)) { const int x = (int)(new_key(kj) & AM); pm |= 1u << x; av[x] = aj; }
            }
        }
        const int xi = (int)(nk & AM);
        if ((pm & ((1u << xi) - 1u)) == 0) {                       // the accepted member: smallest live local index
            int cx = 0;
            const int mc = gtab->mc;
            for (int q = 0; q < mc; ++q) cx |= (int)((nk >> gtab->ctrl_pos[q]) & 1ull) << q;
            const int r = (int)(ps_hash(t ^ 0x9e3779b9u) & (u32)AM);   // the output row this trial draws
            const double2* urow = &gtab->U[((cx << ma) | r) << ma];
            double sr = 0.0, si = 0.0;
            bool any = false;
            for (int c = 0; c < np; ++c) {                         // ascending LOGICAL column index, as the pass
                const int x = gtab->colorder[c];
                if ((pm >> x) & 1u) {
                    const double2 u = urow[x];
                    if (!(u.x == 0.0 && u.y == 0.0)) any = true;
                    cmul_acc(sr, si, u.x, u.y, av[x].x, av[x].y);
                }
            }
            if (any && !(sr == 0.0 && si == 0.0))
                out = ((u64)__double_as_longlong(prob_of(make_double2(sr, si))) >> PS_DROP) + 1ull;
        }
    }
    smp[t] = out;
}

// smp[0..M) ascending; zeros (no output) first.  One warp; thread 0 decides.  mult = 2^ma: outputs a tuple can have.
__global__ void pre_pivot_kernel(const u64* __restrict__ smp, u32 M, u64 n, u32 mult, u64 max_terms, long long slack,
                                 PreCut* __restrict__ pre) {
    if (threadIdx.x != 0) return;
    u32 lo = 0, hi = M;
    while (lo < hi) { const u32 mid = (lo + hi) >> 1; if (smp[mid] == 0) lo = mid + 1; else hi = mid; }
    const u32 z = lo, live = M - z;
    // a trial emits an output >= t with probability C(t) / (mult n), C(t) = outputs with a pattern >= t.
    // js sample points above the floor  =>  C(floor) ~ mult n js / M; ask for max_terms plus 6 sigma.
    const double f = fmin(1.0, (double)max_terms / ((double)mult * (double)n));
    const double js = fmax(1.0, ceil((double)M * f + 6.0 * sqrt(fmax((double)M * f * (1.0 - f), 0.0)) + 8.0) + (double)slack);
    PreCut c;
    c.P_floor = (js >= (double)live) ? 0ull : ((smp[z + (live - (u32)js)] - 1ull) << PS_DROP);
    c.cnt = 0; c.mass_hi = 0.0; c.mass_lo = 0.0;
    *pre = c;
}

// Sums the per-block partials of the pass in block order (fixed order: the same bits every run).  The partials are
// first brought to shared memory by the whole block (one round trip instead of one per partial).
#define PF_MAX 2048
__global__ void __launch_bounds__(1024) pre_finish_kernel(const double* __restrict__ part_mass, const u64* __restrict__ part_cnt,
                                                          u32 nparts, PreCut* __restrict__ pre, u64* __restrict__ d_count) {
    __shared__ double sm[PF_MAX];
    __shared__ u64 sc[PF_MAX];
    for (u32 b = threadIdx.x; b < nparts && b < PF_MAX; b += blockDim.x) { sm[b] = part_mass[b]; sc[b] = part_cnt[b]; }
    __syncthreads();
    if (threadIdx.x != 0) return;
    double hi = 0.0, lo = 0.0;   // double-double running sum
    u64 cnt = 0;
    for (u32 b = 0; b < nparts; ++b) {
        const double x = b < PF_MAX ? sm[b] : part_mass[b];
        const double s = __dadd_rn(hi, x);
        const double bb = __dsub_rn(s, hi);
        const double err = __dadd_rn(__dsub_rn(hi, __dsub_rn(s, bb)), __dsub_rn(x, bb));
        hi = s; lo = __dadd_rn(lo, err);
        cnt += b < PF_MAX ? sc[b] : part_cnt[b];
    }
    const double s = __dadd_rn(hi, lo);
    lo = __dsub_rn(lo, __dsub_rn(s, hi)); hi = s;
    pre->cnt = cnt; pre->mass_hi = hi; pre->mass_lo = lo;
    d_count[2] = cnt;
}

int svk_pre_sample1(const u64* keys, const double2* amps, u64 n, int p, const GateTab* tab, const PendPred& pend, u32 M, u64* smp,
                    cudaStream_t st) {
    pre_sample1_kernel<<<(M + SV_THREADS - 1) / SV_THREADS, SV_THREADS, 0, st>>>(keys, amps, n, p, tab, pend, M, smp);
    return 1;
}
int svk_pre_sample_group(const u64* keys, const double2* amps, u64 n, int p, int ma, const GateTab* tab, const PendPred& pend, u32 M,
                         u64* smp, cudaStream_t st, int p2) {
    pre_sample_group_kernel<<<(M + SV_THREADS - 1) / SV_THREADS, SV_THREADS, 0, st>>>(keys, amps, n, p, ma, tab, pend, M, smp, p2);
    return 1;
}
int svk_pre_pivot(const u64* smp_sorted, u32 M, u64 n, u32 mult, u64 max_terms, long long slack, PreCut* pre, cudaStream_t st) {
    pre_pivot_kernel<<<1, 32, 0, st>>>(smp_sorted, M, n, mult, max_terms, slack, pre);
    return 1;
}
int svk_pre_finish(const double* part_mass, const u64* part_cnt, u32 nparts, PreCut* pre, u64* d_count, cudaStream_t st) {
    pre_finish_kernel<<<1, 1024, 0, st>>>(part_mass, part_cnt, nparts, pre, d_count);
    return 1;
}

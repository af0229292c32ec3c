// Small-state path (SURVEY.md hard part H5; after reordering and fusion the paper's own circuit is
// solved with fewer than 2^5 terms, and its GPU backend shows "a fixed overhead that is apparent at low values of k").
//
// A state of at most SV_SMALL_CAP terms whose gate output also fits SV_SMALL_CAP entries is processed by ONE thread
// block, entirely in shared memory: gate + zero drop + truncation +
// renormalisation in one launch, with the term count kept ON THE DEVICE.  A sequence of such launches needs no host
// round trip: sv_apply_circuit (sv_api.cu) enqueues a whole batch of gates back to back and synchronises once.
//
// The kernel works on STORED keys in the handle's current layout (which it never changes): the gate's qubits are
// given as physical bit positions, the lazy X mask as a pattern `xm` that is XORed into the local indices of U.
//   1. every term finds the other members of its tuple (the terms that differ only in the gate's qubits)
//      by binary search in the sorted key array; the member with the lowest stored pattern OWNS the tuple;
//   2. owners compute the 2^m outputs (columns added in ascending logical index, every operation rounded separately:
//      DESIGN.md D1) into slot (owner rank) * 2^m + row -- or, when every tuple is complete, straight into the
//      positions of the tuple's own members (same keys, same order: nothing to sort);
//   3. truncation, if it can cut: bitonic sort of (p descending, logical key ascending), prefix sums of p in that
//      order, the smallest prefix reaching min_mass * S, capped at max_terms, at least one term; survivors scaled by
//      1/sqrt(kept mass); nothing dropped -> amplitudes untouched (reading R7);
//   4. exact zeros dropped, survivors sorted by stored key (bitonic), written back; count and kept
//      fraction stay on the device.
// If the input or the output does not fit, the kernel sets ctl->status and leaves the state untouched; every later
// launch of the batch then does nothing, and the host continues with the streaming passes from that gate.
// The mass sums here are double-double sums (order independent to ~2^-100), rounded to the same doubles as the exact
// integer sums of the streaming path (D3): threshold, cut, kept mass, scale and kept fraction come out bit for bit the same.
#include "sv_device.cuh"
#include "sv_launch.cuh"

#define SM_T 1024

// bitonic sort of P (power of two) entries by (k1, k2) ascending with payload idx; entries with idx == 0xffff are pads
// and sort last.  TWO: compare k2 on equal k1.
// Pair t of a stage with distance j <= 32 lies inside the 64-entry chunk t / 32: a warp (32 consecutive t per iteration,
// the same t in every stage) then reads only what it wrote itself in the previous stage, so stages with j <= 32 that also
// FOLLOW a stage with j <= 32 are separated by __syncwarp(); only the stages with j >= 64 (10 of the 55 of a 1024-entry
// sort) are bracketed by block barriers.  The sort ends with a block barrier.
template <bool TWO>
__device__ __forceinline__ void bitonic(u64* k1, u64* k2, unsigned short* idx, int P, int A) {
    for (int k = 2; k <= P; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            const int next_j = (j > 1) ? (j >> 1) : ((2 * k <= P) ? k : 1 << 30);   // distance of the stage that follows (none: block barrier)
            for (int t = threadIdx.x; t < (P >> 1); t += A) {
                const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const int l = i | j;
                const bool up = (i & k) == 0;
                const u64 a1 = k1[i], b1 = k1[l];
                const unsigned short ai = idx[i], bi = idx[l];
                u64 a2 = 0, b2 = 0;
                if (TWO) { a2 = k2[i]; b2 = k2[l]; }
                bool a_gt_b;                                   // a sorts after b
                if (ai == 0xffff || bi == 0xffff) a_gt_b = (ai == 0xffff) && (bi != 0xffff);
                else a_gt_b = (a1 > b1) || (TWO && a1 == b1 && a2 > b2);
                const bool b_gt_a = (ai == 0xffff || bi == 0xffff) ? ((bi == 0xffff) && (ai != 0xffff))
                                                                    : ((b1 > a1) || (TWO && a1 == b1 && b2 > a2));
                if (up ? a_gt_b : b_gt_a) {
                    k1[i] = b1; k1[l] = a1; idx[i] = bi; idx[l] = ai;
                    if (TWO) { k2[i] = b2; k2[l] = a2; }
                }
            }
            if (j > 32 || next_j > 32) __syncthreads(); else __syncwarp();
        }
    }
}

// exclusive scan of one int per thread over the block (1024 threads); returns the exclusive prefix, *total the sum
__device__ __forceinline__ int scan1024(int v, int* red, int* total, int A) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nw = A >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    __syncthreads();
    if (lane == 31) red[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const int w = lane < nw ? red[lane] : 0;
        int winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, winc, d); if (lane >= d) winc += t; }
        red[lane] = winc - w;
        if (lane == 31) red[32] = winc;
    }
    __syncthreads();
    *total = red[32];
    return red[warp] + inc - v;
}
// the same for double-double sums (order independent to ~2^-100: the streaming path's exact sums round to the same
// doubles, D3): returns the EXCLUSIVE prefix
__device__ __forceinline__ dd scan1024_excl_dd(dd v, double* red, dd* total, int A) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nw = A >> 5;
    dd inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        dd t; t.hi = __shfl_up_sync(0xffffffffu, inc.hi, d); t.lo = __shfl_up_sync(0xffffffffu, inc.lo, d);
        if (lane >= d) inc = dd_add(inc, t);
    }
    dd exl; exl.hi = __shfl_up_sync(0xffffffffu, inc.hi, 1); exl.lo = __shfl_up_sync(0xffffffffu, inc.lo, 1);
    if (lane == 0) exl = dd_make(0.0);
    __syncthreads();
    if (lane == 31) { red[2 * warp] = inc.hi; red[2 * warp + 1] = inc.lo; }
    __syncthreads();
    if (warp == 0) {
        dd w = dd_make(0.0);
        if (lane < nw) { w.hi = red[2 * lane]; w.lo = red[2 * lane + 1]; }
        dd winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            dd t; t.hi = __shfl_up_sync(0xffffffffu, winc.hi, d); t.lo = __shfl_up_sync(0xffffffffu, winc.lo, d);
            if (lane >= d) winc = dd_add(winc, t);
        }
        dd wex; wex.hi = __shfl_up_sync(0xffffffffu, winc.hi, 1); wex.lo = __shfl_up_sync(0xffffffffu, winc.lo, 1);
        if (lane == 0) wex = dd_make(0.0);
        __syncwarp();
        red[2 * lane] = wex.hi; red[2 * lane + 1] = wex.lo;
        if (lane == 31) { red[64] = winc.hi; red[65] = winc.lo; }
    }
    __syncthreads();
    total->hi = red[64]; total->lo = red[65];
    dd pre; pre.hi = red[2 * warp]; pre.lo = red[2 * warp + 1];
    return dd_add(pre, exl);
}

__global__ void __launch_bounds__(SM_T, 1) small_gate_kernel(u64* __restrict__ keys, double2* __restrict__ amps, SmallCtl* __restrict__ ctl,
                                                             const SmallGate* __restrict__ gates, int n_gates, KeyMap km, u64 max_terms,
                                                             double min_mass, double* __restrict__ kept_out, u64 cap) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* ia = reinterpret_cast<double2*>(smem_raw);
    double2* oa = ia + SV_SMALL_CAP;
    u64* ik = reinterpret_cast<u64*>(oa + SV_SMALL_CAP);
    u64* ok = ik + SV_SMALL_CAP;
    unsigned short* oidx = reinterpret_cast<unsigned short*>(ok + SV_SMALL_CAP);
    unsigned short* oelem = oidx + SV_SMALL_CAP;       // element index of the owner of every tuple
    __shared__ double2 sU[256];
    __shared__ int s_pos[SV_MAX_M];
    __shared__ int red[33];
    __shared__ double redd[66];
    __shared__ int s_flag;
    const int tid = threadIdx.x;
    const int A = blockDim.x;                         // the host sizes the block to the work it expects (a barrier among few warps is cheap)
    const u64 n64 = ctl->count;
    if (n64 > SV_SMALL_CAP) { if (tid == 0) { ctl->status = 1; ctl->fail_gate = 0; ctl->done_gates = 0; } return; }
    int n = (int)n64;
    // The state is loaded ONCE and stays in shared memory for the whole batch of gates: no launch, no global round trip
    // and no reload between two gates.
    for (int e = tid; e < n; e += A) { ik[e] = keys[e]; ia[e] = amps[e]; }
    int done = 0, failed = 0;
    u64 last_pre = 0;
    for (int gi = 0; gi < n_gates; ++gi) {
    const SmallGate* gate = gates + gi;
    const int m = gate->m, xm = gate->xm;
    const int NP = 1 << m;
    __syncthreads();                                  // the previous gate is complete (state in ik / ia, tables free)
    for (int i = tid; i < 256; i += A) sU[i] = gate->U[i];
    if (tid < SV_MAX_M) s_pos[tid] = gate->pos[tid];
    __syncthreads();
    u64 mask = 0;
    for (int j = 0; j < m; ++j) mask |= 1ull << s_pos[j];
    auto scatter = [&](int pat) { u64 v = 0; for (int j = 0; j < m; ++j) v |= (u64)((pat >> j) & 1) << s_pos[j]; return v; };
    auto find = [&](u64 key) {                        // index of key in ik[0..n), or -1
        int lo = 0, hi = n;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (ik[mid] < key) lo = mid + 1; else hi = mid; }
        return (lo < n && ik[lo] == key) ? lo : -1;
    };

    // ---- 1. owners.  Every step is spread over all active threads (a few threads walking whole tuples serially would
    // leave the other warps waiting at the barriers) ----
    // 1a: element e is NOT an owner iff some member with a lower stored pattern exists: one search per (element, pattern)
    for (int e = tid; e < n; e += A) oidx[e] = 0;
    __syncthreads();
    for (int t = tid; t < (n << m); t += A) {
        const int e = t >> m, y = t & (NP - 1);
        const u64 k = ik[e];
        int cs = 0;
        for (int j = 0; j < m; ++j) cs |= (int)((k >> s_pos[j]) & 1ull) << j;
        if (y < cs && find((k & ~mask) | scatter(y)) >= 0) oidx[e] = 1;      // (racing writers all write 1)
    }
    __syncthreads();
    // 1b: owner ranks in key order (thread t takes the elements t * per .. consecutively: one scan)
    const int per = (n + A - 1) / A;                  // <= 4
    int cown = 0;
    for (int i = 0; i < per; ++i) { const int e = tid * per + i; if (e < n && !oidx[e]) ++cown; }
    int n_owners;
    int orank = scan1024(cown, red, &n_owners, A);
    const long long n_slots = (long long)n_owners << m;
    if (n_slots > SV_SMALL_CAP) { failed = 1; break; }
    for (int i = 0; i < per; ++i) { const int e = tid * per + i; if (e < n && !oidx[e]) oelem[orank++] = (unsigned short)e; }
    const bool in_place = (n_slots == n);             // every tuple complete: the outputs take the members' own positions
    const int ns = (int)n_slots;                      // output slots (exact zeros among them)
    __syncthreads();
    // 1c: the members of every owner's tuple: memtab[owner * 2^m + stored pattern] = element index, 0xffff if absent
    unsigned short* memtab = oidx;
    for (int t = tid; t < ns; t += A) {
        const int o = t >> m, y = t & (NP - 1);
        const int f = find((ik[oelem[o]] & ~mask) | scatter(y));
        memtab[t] = (unsigned short)(f < 0 ? 0xffff : f);
    }
    __syncthreads();
    // ---- 2. outputs: one task per (tuple, row) ----
    int nz_mine = 0;
    for (int t = tid; t < ns; t += A) {
        const int o = t >> m, rs = t & (NP - 1), r = rs ^ xm;     // r, c: TRUE local patterns; stored pattern = true ^ xm
        const u64 base = ik[oelem[o]] & ~mask;
        double sr = 0.0, si = 0.0;
        for (int c = 0; c < NP; ++c) {                             // ascending logical column (D1); absent members skipped
            const unsigned short mi = memtab[(o << m) | (c ^ xm)];
            if (mi != 0xffff) {
                const double2 a = ia[mi];
                const double2 u = sU[r * NP + c];
                cmul_acc(sr, si, u.x, u.y, a.x, a.y);
            }
        }
        const int slot = in_place ? (int)memtab[t] : t;
        ok[slot] = base | scatter(rs);
        oa[slot] = make_double2(sr, si);
        nz_mine += (sr == 0.0 && si == 0.0) ? 0 : 1;
    }
    int n_pre;                                        // nonzero outputs = terms after the gate
    scan1024(nz_mine, red, &n_pre, A);
    // (capacity bounds the terms that exist at any instant, a gate's output before its cut included: the streaming path
    // reports SV_ERR_CAPACITY for this gate)
    if ((u64)n_pre > cap) { failed = 1; break; }
    __syncthreads();

    // ---- 3. truncation ----
    const bool needK = max_terms != 0 && max_terms < (u64)n_pre, needM = min_mass < 1.0;
    double kept_fraction = 1.0;
    if ((needK || needM) && n_pre > 0) {
        int P = 2; while (P < ns) P <<= 1;
        u64* s1 = ik;                                               // ~pattern of p  (the input arrays are free now)
        u64* s2 = reinterpret_cast<u64*>(ia);                       // logical key
        for (int e = tid; e < P; e += A) {
            if (e < ns && !(oa[e].x == 0.0 && oa[e].y == 0.0)) {
                s1[e] = ~(u64)__double_as_longlong(prob_of(oa[e]));
                s2[e] = logical_key(ok[e], km);
                oidx[e] = (unsigned short)e;
            } else { s1[e] = ~0ull; s2[e] = ~0ull; oidx[e] = 0xffff; }
        }
        __syncthreads();
        bitonic<true>(s1, s2, oidx, P, A);
        // masses in sorted order: thread t holds the ranks t * rper .. (consecutive)
        const int rper = (n_pre + A - 1) / A;
        dd loc = dd_make(0.0);
        for (int q = 0; q < rper; ++q) {
            const int rnk = tid * rper + q;
            if (rnk < n_pre) loc = dd_add(loc, dd_make(__longlong_as_double((long long)~s1[rnk])));
        }
        dd S;
        const dd excl = scan1024_excl_dd(loc, redd, &S, A);
        // j_mass: the smallest j with cum_j >= min_mass * S (the threshold rounded once, as the streaming path takes it)
        const dd thr = dd_make(__dmul_rn(min_mass, S.hi));
        int jm_local = 0x7fffffff;
        if (needM) {
            dd cum = excl;
            for (int q = 0; q < rper; ++q) {
                const int rnk = tid * rper + q;
                if (rnk < n_pre) {
                    cum = dd_add(cum, dd_make(__longlong_as_double((long long)~s1[rnk])));
                    if (dd_ge(cum, thr) && jm_local == 0x7fffffff) jm_local = rnk + 1;
                }
            }
        }
        if (tid == 0) s_flag = 0x7fffffff;
        __syncthreads();
        if (jm_local != 0x7fffffff) atomicMin(&s_flag, jm_local);
        __syncthreads();
        int j = n_pre;
        if (needM && s_flag != 0x7fffffff) j = s_flag;
        if (max_terms != 0 && (u64)j > max_terms) j = (int)max_terms;
        if (j < 1) j = 1;
        __syncthreads();
        if (j < n_pre) {
            {   // kept mass = cum_j (held by the thread that owns rank j - 1)
                dd cum = excl;
                for (int q = 0; q < rper; ++q) {
                    const int rnk = tid * rper + q;
                    if (rnk < n_pre) {
                        cum = dd_add(cum, dd_make(__longlong_as_double((long long)~s1[rnk])));
                        if (rnk + 1 == j) redd[0] = cum.hi;
                    }
                }
            }
            __syncthreads();
            const double kept = redd[0];
            const double scale = __ddiv_rn(1.0, __dsqrt_rn(kept));
            kept_fraction = __ddiv_rn(kept, S.hi);
            for (int rnk = tid; rnk < n_pre; rnk += A) {
                const int e = oidx[rnk];
                if (rnk < j) { oa[e].x = __dmul_rn(oa[e].x, scale); oa[e].y = __dmul_rn(oa[e].y, scale); }
                else { oa[e].x = 0.0; oa[e].y = 0.0; }                 // dropped: squeezed out with the exact zeros below
            }
            __syncthreads();
        }
    }

    // ---- 4. zero drop (stable compaction of the slots), order by stored key, write back ----
    int n_final;
    {
        const int sper = (ns + A - 1) / A;
        int c = 0;
        for (int q = 0; q < sper; ++q) { const int e = tid * sper + q; if (e < ns && !(oa[e].x == 0.0 && oa[e].y == 0.0)) ++c; }
        int w = scan1024(c, red, &n_final, A);
        if (in_place) {       // the slots are in key order already
            for (int q = 0; q < sper; ++q) {
                const int e = tid * sper + q;
                if (e < ns && !(oa[e].x == 0.0 && oa[e].y == 0.0)) { ik[w] = ok[e]; ia[w] = oa[e]; ++w; }
            }
        } else {              // sort the survivors only
            u64* s1 = ik;
            for (int q = 0; q < sper; ++q) {
                const int e = tid * sper + q;
                if (e < ns && !(oa[e].x == 0.0 && oa[e].y == 0.0)) { s1[w] = ok[e]; oidx[w] = (unsigned short)e; ++w; }
            }
            int P = 2; while (P < n_final) P <<= 1;
            __syncthreads();
            for (int e = n_final + tid; e < P; e += A) { s1[e] = ~0ull; oidx[e] = 0xffff; }
            __syncthreads();
            bitonic<false>(s1, nullptr, oidx, P, A);
            for (int e = tid; e < n_final; e += A) ia[e] = oa[oidx[e]];          // (the sorted keys already sit in ik)
        }
    }
    if (tid == 0 && kept_out) kept_out[gi] = kept_fraction;
    n = n_final;
    last_pre = (u64)n_pre;
    done = gi + 1;
    }   // gates
    __syncthreads();
    // write the state back (on a gate that did not fit: the state before that gate, untouched in ik / ia)
    for (int e = tid; e < n; e += A) { keys[e] = ik[e]; amps[e] = ia[e]; }
    if (tid == 0) {
        ctl->count = (u64)n;
        ctl->n_pre = last_pre;
        ctl->done_gates = done;
        ctl->status = failed;
        ctl->fail_gate = failed ? done : -1;
    }
}

size_t svk_small_smem() { return (size_t)SV_SMALL_CAP * (16 + 16 + 8 + 8 + 2 + 2); }

// `threads`: block size (a multiple of 32 in 256..1024), from the host's bound on the work of a gate
int svk_small_gates(u64* keys, double2* amps, SmallCtl* ctl, const SmallGate* gates, int n_gates, KeyMap km, u64 max_terms, double min_mass,
                    double* kept_out, u64 cap, int threads, cudaStream_t st) {
    static bool attr[SV_MAX_DEV];
    const size_t smem = svk_small_smem();
    sv_set_smem_once(small_gate_kernel, smem, attr);
    if (threads < 256) threads = 256;
    if (threads > SM_T) threads = SM_T;
    threads = (threads + 31) & ~31;
    small_gate_kernel<<<1, threads, smem, st>>>(keys, amps, ctl, gates, n_gates, km, max_terms, min_mass, kept_out, cap);
    return 1;
}

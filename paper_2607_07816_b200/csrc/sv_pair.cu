// Single-bit pass (SURVEY.md rows a-3 .. a-7 for gates with ONE active bit, and the pure bit
// moves of wider gates).  PAPER.md:110-120.
//
// Keys are stored ascending in the physical bit order.  Moving physical bit p to the LSB
// is, inside every block of keys that agree above p, a merge of the run with bit p = 0
// ("A") and the run with bit p = 1 ("B") by the remaining bits.  Over a whole tile (a
// merge-path slice of the state, see find_splits) the A terms of all its blocks, taken in
// stored order, are ascending in the key with bit p cleared, and so are the B terms: the
// pass is ONE two-way merge of two sorted sequences A* and B* per tile.
//
//   load      the tile's (up to three) contiguous pieces; a truncation left pending by
//             sv_truncate is applied here (dropped terms load as 0+0i, survivors are scaled);
//             terms are placed in shared memory partitioned into A* | B*;
//   split     every thread finds where its VT consecutive OUTPUT positions start in A* and
//             B* (merge path: one binary search per thread, not per term);
//   merge     VT sequential merge steps per thread.  Partners (the terms
//             that differ only in the gate's qubit) meet as neighbours: the A member leads,
//             the 2x2 mat-vec runs on the spot, exact zeros are dropped
//             (PAPER.md:13);
//   write     block scan + decoupled look-back give the output offsets; the outputs are
//             staged in shared memory in output order and stored with coalesced writes:
//             sorted, unique keys by construction.
#include "sv_device.cuh"

#define BP_VT 4
#define BP_TILE (SV_THREADS * BP_VT)      // 1024 terms per tile
#define BP_TNOM (BP_TILE - 2)             // nominal tile (boundaries are pulled back to a tuple start)
#define BP_WARPS (SV_THREADS / 32)

__device__ __forceinline__ bool pend_keep(const PendPred& pd, u64 stored_key, double2 a) {
    const u64 pat = (u64)__double_as_longlong(prob_of(a));
    if (pat > pd.PT) return true;
    if (pat < pd.PT) return false;
    if (pd.KT == ~0ull) return true;
    return logical_key(stored_key, pd.km) <= pd.KT;
}

template <bool PAIR>
__global__ void __launch_bounds__(SV_THREADS, 4) bitpass_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                                u64* __restrict__ kout, double2* __restrict__ aout, int p,
                                                                const GateTab* __restrict__ gtab, PendPred pd,
                                                                const TileDesc* __restrict__ desc, u64* status,
                                                                u64* d_count, u64 cap, u32 ntiles) {
    constexpr int OUTCAP = PAIR ? 2 * BP_TILE : BP_TILE;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* sta = reinterpret_cast<double2*>(smem_raw);      // staged outputs; its front doubles as the input tile
    u64* stk = reinterpret_cast<u64*>(sta + OUTCAP);
    double2* sa = sta;
    u64* sk = stk;
    __shared__ int red[BP_WARPS + 2];
    __shared__ int wc[BP_VT][BP_WARPS];
    __shared__ int s_nA;
    __shared__ u64 s_base;
    __shared__ double2 sU[64];      // [cx][xr][xc], ma = 1: up to 8 control patterns x 4
    __shared__ int s_cpos[SV_MAX_M], s_mc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // Tiles are taken in blockIdx order: a block only ever waits on lower-numbered blocks,
    // which the hardware scheduler has already started.
    const u32 tile = blockIdx.x;
    if (PAIR) {
        if (tid < 64) sU[tid] = gtab->U[tid];
        if (tid < SV_MAX_M) s_cpos[tid] = gtab->ctrl_pos[tid];
        if (tid == 0) s_mc = gtab->mc;
    }
    const TileDesc d0 = desc[tile], d1 = desc[tile + 1];
    const bool oneblock = (d0.e == d1.e);
    u64 ps0, ps1, ps2; int l0, l1, l2;
    if (oneblock) { ps0 = d0.ia; l0 = (int)(d1.ia - d0.ia); ps1 = d0.ib; l1 = (int)(d1.ib - d0.ib); ps2 = 0; l2 = 0; }
    else { ps0 = d0.ia; l0 = (int)(d0.mid - d0.ia); ps1 = d0.ib; l1 = (int)(d1.ia - d0.ib); ps2 = d1.mid; l2 = (int)(d1.ib - d1.mid); }
    const int cnt = min(BP_TILE, l0 + l1 + l2);
    const u64 bit = 1ull << p;
    int nA;
    {   // coalesced loads of the contiguous pieces, all issued before any is used
        u64 lk[BP_VT]; double2 la[BP_VT];
#pragma unroll
        for (int r = 0; r < BP_VT; ++r) {
            const int e = tid + r * SV_THREADS;
            lk[r] = 0; la[r] = make_double2(0.0, 0.0);
            if (e < cnt) {
                const u64 g = e < l0 ? ps0 + e : (e < l0 + l1 ? ps1 + (e - l0) : ps2 + (e - l0 - l1));
                lk[r] = ld_stream_u64(kin + g);
                la[r] = ld_stream_d2(ain + g);
            }
        }
        if (pd.active) {
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                if (tid + r * SV_THREADS < cnt) {
                    if (pend_keep(pd, lk[r], la[r])) { la[r].x = __dmul_rn(la[r].x, pd.scale); la[r].y = __dmul_rn(la[r].y, pd.scale); }
                    else { la[r].x = 0.0; la[r].y = 0.0; }
                }
            }
        }
        if (oneblock) {   // piece 0 is all A, piece 1 all B: the load order is already A* | B*
            nA = l0;
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const int e = tid + r * SV_THREADS;
                if (e < cnt) { sk[e] = lk[r] & ~bit; sa[e] = la[r]; }
            }
        } else {          // stable partition by bit p (the load order is the stored order)
            u32 balA[BP_VT];
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const bool isA = (tid + r * SV_THREADS < cnt) && !(lk[r] & bit);
                balA[r] = __ballot_sync(0xffffffffu, isA);
                if (lane == 0) wc[r][warp] = __popc(balA[r]);
            }
            __syncthreads();
            if (warp == 0) {   // lane = r * 8 + warp: exclusive scan of the 32 counts in load order
                const int c = wc[lane >> 3][lane & 7];
                int inc = c;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                wc[lane >> 3][lane & 7] = inc - c;
                if (lane == 31) s_nA = inc;
            }
            __syncthreads();
            nA = s_nA;
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const int e = tid + r * SV_THREADS;
                if (e < cnt) {
                    const int aBefore = wc[r][warp] + __popc(balA[r] & ((1u << lane) - 1u));
                    const int slot = (lk[r] & bit) ? nA + (e - aBefore) : aBefore;
                    sk[slot] = lk[r] & ~bit; sa[slot] = la[r];
                }
            }
        }
    }
    __syncthreads();
    const int nB = cnt - nA;
    const u64* skB = sk + nA;
    const double2* saB = sa + nA;

    // merge-path split of this thread's first output position
    const int diag = min(tid * BP_VT, cnt);
    int i, j;
    {
        int lo = max(0, diag - nB), hi = min(diag, nA);
        while (lo < hi) {   // A first on ties
            const int mid = (lo + hi) >> 1;
            if (sk[mid] <= skB[diag - 1 - mid]) lo = mid + 1; else hi = mid;
        }
        i = lo; j = diag - lo;
    }
    const int endpos = min(diag + BP_VT, cnt);
    int pos = diag;
    const u64 himask = (p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    // keys with bit p cleared never equal ~0: safe sentinels for an exhausted side
    u64 ka = (i < nA) ? sk[i] : ~0ull, kb = (j < nB) ? skB[j] : ~0ull;
    u64 ok[BP_VT];
    double o0r[BP_VT], o0i[BP_VT], o1r[BP_VT], o1i[BP_VT];
    u32 fl = 0;     // two flag bits per step
    int nout = 0;
    if (PAIR && pos < endpos && j < nB && i > 0 && sk[i - 1] == kb) {   // this B belongs to the previous thread's tuple
        ++j; ++pos;
        kb = (j < nB) ? skB[j] : ~0ull;
    }
#pragma unroll
    for (int v = 0; v < BP_VT; ++v) {
        ok[v] = 0; o0r[v] = o0i[v] = o1r[v] = o1i[v] = 0.0;
        if (pos < endpos) {
            const bool takeA = ka <= kb;
            const u64 k = takeA ? ka : kb;
            const u64 nk = (k & himask) | ((k & lowmask) << 1);     // new layout, LSB = 0
            if (PAIR) {
                double2 a, pa = make_double2(0.0, 0.0);
                bool has_partner = false;
                if (takeA) {
                    a = sa[i]; ++i; ++pos;
                    has_partner = (kb == k);
                    if (has_partner) { pa = saB[j]; ++j; ++pos; kb = (j < nB) ? skB[j] : ~0ull; }
                    ka = (i < nA) ? sk[i] : ~0ull;
                } else {
                    a = saB[j]; ++j; ++pos;
                    kb = (j < nB) ? skB[j] : ~0ull;
                }
                int cx = 0;
                const int mc = s_mc;
                for (int q = 0; q < mc; ++q) cx |= (int)((nk >> s_cpos[q]) & 1ull) << q;
                const double2* u = &sU[cx << 2];                    // u[xr * 2 + xc]
                double r0 = 0.0, m0 = 0.0, r1 = 0.0, m1 = 0.0;
                if (takeA) {
                    cmul_acc(r0, m0, u[0].x, u[0].y, a.x, a.y);
                    cmul_acc(r1, m1, u[2].x, u[2].y, a.x, a.y);
                    if (has_partner) {
                        cmul_acc(r0, m0, u[1].x, u[1].y, pa.x, pa.y);
                        cmul_acc(r1, m1, u[3].x, u[3].y, pa.x, pa.y);
                    }
                } else {
                    cmul_acc(r0, m0, u[1].x, u[1].y, a.x, a.y);
                    cmul_acc(r1, m1, u[3].x, u[3].y, a.x, a.y);
                }
                const u32 f0 = !(r0 == 0.0 && m0 == 0.0), f1 = !(r1 == 0.0 && m1 == 0.0);
                ok[v] = nk; o0r[v] = r0; o0i[v] = m0; o1r[v] = r1; o1i[v] = m1;
                fl |= (f0 | (f1 << 1)) << (2 * v);
                nout += (int)(f0 + f1);
            } else {
                const double2 a = takeA ? sa[i] : saB[j];
                if (takeA) { ++i; ka = (i < nA) ? sk[i] : ~0ull; } else { ++j; kb = (j < nB) ? skB[j] : ~0ull; }
                ++pos;
                const u32 f0 = !(a.x == 0.0 && a.y == 0.0);
                ok[v] = nk | (takeA ? 0ull : 1ull); o0r[v] = a.x; o0i[v] = a.y;
                fl |= f0 << (2 * v);
                nout += (int)f0;
            }
        }
    }
    int total;
    const int excl = block_excl_scan(nout, red, &total);   // its barriers also retire every read of the input tile
    if (tid < 32) {
        const u64 ex = lookback_exclusive_warp(status, tile, (u64)total);
        if (tid == 0) {
            s_base = ex;
            if (tile == ntiles - 1) *d_count = ex + (u64)total;
        }
    }
    {   // stage the outputs in output order (the staging area aliases the consumed input tile)
        int off = excl;
#pragma unroll
        for (int v = 0; v < BP_VT; ++v) {
            const u32 f = (fl >> (2 * v)) & 3u;
            if (f & 1u) { stk[off] = ok[v]; sta[off] = make_double2(o0r[v], o0i[v]); ++off; }
            if (PAIR && (f & 2u)) { stk[off] = ok[v] | 1ull; sta[off] = make_double2(o1r[v], o1i[v]); ++off; }
        }
    }
    __syncthreads();
    const u64 base = s_base;
    for (int idx = tid; idx < total; idx += SV_THREADS) {
        const u64 g = base + (u64)idx;
        if (g < cap) { st_stream_u64(kout + g, stk[idx]); st_stream_d2(aout + g, sta[idx]); }
    }
}

template <bool PAIR>
static void launch_bitpass(const u64* kin, const double2* ain, u64* kout, double2* aout, int p, const GateTab* tab,
                           const PendPred& pend, TileDesc* desc, u64* status, u64* d_count, u64 cap, u32 ntiles, cudaStream_t st) {
    const size_t smem = (size_t)(PAIR ? 2 : 1) * BP_TILE * 24;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(bitpass_kernel<PAIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr = true; }
    bitpass_kernel<PAIR><<<ntiles, SV_THREADS, smem, st>>>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles);
}

int svk_bitpass(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int pair,
                const GateTab* tab, const PendPred& pend, TileDesc* desc, u64* status, u32* tile_counter,
                u64* d_count, u64 cap, cudaStream_t st, cudaEvent_t e0, cudaEvent_t e1) {
    (void)tile_counter;
    if (n == 0) { cudaMemsetAsync(d_count, 0, sizeof(u64), st); return 0; }
    const u32 ntiles = (u32)((n + BP_TNOM - 1) / BP_TNOM);
    cudaMemsetAsync(status, 0, (size_t)ntiles * sizeof(u64), st);
    int launches = svk_find_splits(kin, n, p, 0, BP_TNOM, ntiles, desc, st);
    if (e0) cudaEventRecord(e0, st);
    if (pair) launch_bitpass<true>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st);
    else launch_bitpass<false>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st);
    if (e1) cudaEventRecord(e1, st);
    return launches + 1;
}

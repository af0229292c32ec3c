// Final pass of a DENSE gate with MA >= 2 active bits -- every entry of U nonzero, no control-like bit (Haar SU(4),
// Haar 8x8, 16x16, fused blocks): SURVEY.md rows a-4 .. a-7.
//
// Front end as in sv_group.cu (persistent blocks, the next tile landing by bulk copies, A* | B* partition, one
// merge-path split per thread, the tile left in shared memory in its NEW order where the members of a tuple --
// the terms that differ only in the gate's qubits -- are neighbours), except that dead entries and the
// terms a pending truncation drops are squeezed out while the tile is partitioned: behind the front end every
// element of the tile is a live term.
//
// Back end.  U has no zero entry, so every tuple yields exactly 2^MA candidate outputs: no owner table, no per-tuple row
// masks.  ONE THREAD PER TUPLE computes all 2^MA rows in registers (columns added in ascending logical
// index, every operation rounded separately: DESIGN.md D1): the tuple's members are read once, U comes from shared memory
// with the lanes of a warp spread over its columns (conflict free), and a round of 256 * TPR tuples costs no per-candidate
// bookkeeping.
//   two calls (PRE = false): the tile's output count is known before any arithmetic; a thread's 2^MA rows are consecutive
//     outputs and go out straight from registers with 256-bit stores (an exact cancellation is written as a counted dead
//     entry); the look-back resolves behind the first round's arithmetic.
//   fused apply + truncate (PRE = true): every candidate is computed ONCE, tested against the floor of the cut that
//     follows (sv_presample.cu); survivors are ranked by warp scans + one block scan per round and staged in output
//     order in shared memory; the tile's total is published when its last round is done and the staged outputs stay
//     PARKED while the block prepares its next tile, then stored coalesced.  A tile with more survivors than the
//     staging buffer holds (a heavy region of the state) resolves its look-back at once and computes its candidates a
//     second time, storing them directly.
#include "sv_tile.cuh"
#include "sv_launch.cuh"
#include <type_traits>

#ifndef DP_NOPRE_BLOCKS
#define DP_NOPRE_BLOCKS 4                  // resident blocks per SM of the two-call variant (ma <= 3): 64 registers, ~51 KB of shared memory
#endif
// The tile's key array sk is addressed through an XOR swizzle of the entry index with its 128-byte row (16 keys per row), as
// the staging arrays of sv_pair.cu: threads that own a few CONSECUTIVE entries each (the merges write 4 per thread, read ~2
// apart per lane) would otherwise hit the same banks 4 to 8 ways -- measured: a third of the kernel's shared-memory wavefronts
// were such replays and the shared-memory pipe its busiest unit (72 %).
#define DK(x) ((x) ^ (((x) >> 4) & 15))

#ifndef DP_STAGE
#define DP_STAGE 2048                      // PRE: staged survivors per tile (about twice the mean at the cap)
#endif

// TWO: the pass moves TWO bits (p > p2) to the two least-significant positions at once.  A tile (TileDesc2, find_splits2 in
// sv_gate.cu) is then up to seven contiguous pieces of the input; its live entries are partitioned into the four classes of
// (bH, bL) -- each sorted by the rest of the key -- and merged in two levels: the bL = 0 / 1 classes of either bH (two
// merges side by side, one merge-path split per thread), then the two results by bH.  The state comes out as the two
// single-bit passes (p, then p2 + 1) would leave it, without the intermediate trip through HBM.
#define DP_MAXPIECES 8
template <int MA, bool PRE, bool TWO>
__global__ void __launch_bounds__(SV_THREADS, (PRE || MA > 3) ? 2 : DP_NOPRE_BLOCKS) densepass_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                                            u64* __restrict__ kout, double2* __restrict__ aout, int p,
                                                                            const GateTab* __restrict__ gtab, PendPred pd,
                                                                            const TileDesc* __restrict__ desc, u64* status,
                                                                            u64* d_count, u64 cap, u32 ntiles, const PreCut* __restrict__ pre,
                                                                            double* __restrict__ pre_mass, u64* __restrict__ pre_cnt,
                                                                            int maybe_dead, int p2) {
    constexpr int NP = 1 << MA;
    constexpr int LKX = TWO ? 16 : 8;            // over-fetched keys the landing array has room for (two per piece)
    constexpr u64 AM = (u64)NP - 1;
    constexpr int TPR = NP >= 8 ? 1 : 8 / NP;   // tuples per thread and round
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // Amplitudes never move inside shared memory: a tile's amplitudes stay where the bulk copies put them (two landing
    // buffers used in turns, the next tile landing in the other one) and the partition and the merges move (key, 16-bit
    // landing index) pairs only; the tuple arithmetic reads each amplitude once, by its index.
    double2* La0 = reinterpret_cast<double2*>(smem_raw);
    double2* La1 = La0 + BP_TILE;
    u64* Lk = reinterpret_cast<u64*>(La1 + BP_TILE);
    u64* sk = Lk + BP_TILE + LKX;
    unsigned short* tst = reinterpret_cast<unsigned short*>(sk + BP_TILE);   // first member of every tuple (+ sentinel)
    unsigned short* si = tst + BP_TILE + 8;                                  // landing index of the entry whose key sits in sk (same slot, unswizzled)
    double2* stg_a = reinterpret_cast<double2*>(si + BP_TILE);               // PRE only: staged survivors, output order
    u64* stg_k = reinterpret_cast<u64*>(stg_a + DP_STAGE);
    __shared__ int wcA[BP_VT][BP_WARPS], wcB[BP_VT][BP_WARPS];
    __shared__ int s_nA, s_nB, s_nt;
    __shared__ u64 s_last[BP_WARPS];        // last merged key of every warp (tuple starts across warps)
    __shared__ int wtot[2][BP_WARPS];
    __shared__ u64 s_desc[2][TWO ? 16 : 8];
    __shared__ int s_pcum[2][TWO ? DP_MAXPIECES + 1 : 1], s_pko[2][TWO ? DP_MAXPIECES : 1];   // TWO: first load-order index of every piece (+ total), key slot offset
    __shared__ int wc4[TWO ? 4 : 1][BP_VT][BP_WARPS], s_n4[4];                                 // TWO: class counts per (round, warp); class totals
    __shared__ u64 s_base;
    __shared__ __align__(8) u64 s_bar;   // mbarrier of the landing bulk copies
    __shared__ double2 Us[NP * NP];          // Us[r * NP + x] = U[r][x] (physical patterns): lanes differ in x -> different banks
    __shared__ int s_col[16];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 lt = (1u << lane) - 1u;
    const bool mv = p >= 0;
    const u64 Pf = PRE ? pre->P_floor : 0ull;
    double dmass = 0.0;     // PRE: mass and number of the outputs this thread left out (below the floor)
    u32 dcnt = 0;
    u32 n_dead = 0;         // !PRE: exact cancellations written as dead entries

    if (tid < NP * NP) Us[tid] = gtab->U[tid];
    if (tid < 16) s_col[tid] = gtab->colorder[tid];
    __syncthreads();
    u64 colpack = 0;        // logical column t -> physical pattern, 4 bits each
#pragma unroll
    for (int t = 0; t < NP; ++t) colpack |= (u64)(s_col[t] & 15) << (4 * t);
    bool col_ident = true;
#pragma unroll
    for (int t = 0; t < NP; ++t) col_ident = col_ident && (s_col[t] == t);

    const u64 bit = mv ? (1ull << p) : 0ull;
    const u64 himask = (!mv || p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    // TWO: stored key (high, bH, mid, bL, low) -> (high, mid, low, 0, 0)
    const u64 bit2 = TWO ? (1ull << p2) : 0ull;
    const u64 midmask = TWO ? ((bit - 1) & ~((bit2 << 1) - 1)) : 0ull, lowmask2 = TWO ? (bit2 - 1) : 0ull;
    u64* gstat = status + ntiles;
    // parked tile (PRE): its staged outputs wait for the look-back while the next tile is prepared
    bool pk_valid = false;  // uniform over the block
    u32 pk_tile = 0; int pk_total = 0;

    // The tile lands by bulk copies (TMA): one thread arms the barrier and issues up to six copies (sv_tile.cuh).
    auto issue_loads = [&](const Pieces3& q, double2* La) {
        if (tid == 0) land_tile_bulk(q, kin, ain, Lk, La, &s_bar);
    };
    // TWO, called by ONE thread: w = the tile's entry of the piece table (make_pieces2 in sv_gate.cu: start index and length
    // of its up to seven contiguous pieces of the input).  Fills the table the pick-up reads (s_pcum / s_pko[slot]) and
    // issues the bulk copies.  A key piece that starts at an odd index is fetched from the even index before it (sv_tile.cuh).
    auto issue_loads2 = [&](const u64* w, int slot, double2* La) {
        u64 ps[DP_MAXPIECES]; int pl[DP_MAXPIECES];
        int np = 0;
#pragma unroll
        for (int q = 0; q < DP_MAXPIECES; ++q) {
            ps[q] = w[q];
            pl[q] = (int)(u32)(w[DP_MAXPIECES + q / 2] >> (32 * (q & 1)));
            np += pl[q] ? 1 : 0;
        }
        int cum = 0, slots = 0;
        u32 bytes = 0;
#pragma unroll
        for (int q = 0; q < DP_MAXPIECES; ++q) {     // (unused pieces have length 0: they start where the tile ends)
            const int o = (int)(ps[q] & 1ull), c = pl[q] ? ((pl[q] + o + 1) & ~1) : 0;
            s_pcum[slot][q] = cum; s_pko[slot][q] = pl[q] ? (slots + o - cum) : 0;
            bytes += (u32)c * 8u + (u32)pl[q] * 16u;
            cum += pl[q]; slots += c;
        }
        s_pcum[slot][DP_MAXPIECES] = cum;
        SV_CHK(np <= DP_MAXPIECES && cum <= BP_TILE && slots <= BP_TILE + LKX);
        fence_proxy_async_smem();
        mbar_expect_tx(&s_bar, bytes);
        cum = 0; slots = 0;
#pragma unroll
        for (int q = 0; q < DP_MAXPIECES; ++q) {
            if (pl[q]) {
                const int o = (int)(ps[q] & 1ull), c = (pl[q] + o + 1) & ~1;
                bulk_g2s(Lk + slots, kin + (ps[q] & ~1ull), (u32)c * 8u, &s_bar);
                bulk_g2s(La + cum, ain + ps[q], (u32)pl[q] * 16u, &s_bar);
                cum += pl[q]; slots += c;
            }
        }
    };
    if (tid == 0) { mbar_init(&s_bar, 1); fence_proxy_async_smem(); }
    u32 bar_phase = 0;
    auto flush_parked = [&]() {   // resolve the parked tile's look-back, store its staged outputs coalesced
        if (tid < 32) {
            const u64 ex = lookback_exclusive_2level<false>(status, gstat, pk_tile, ntiles, (u64)pk_total);
            if (tid == 0) {
                s_base = ex;
                if (pk_tile == ntiles - 1) d_count[0] = ex + (u64)pk_total;
            }
        }
        __syncthreads();
        const u64 base = s_base;
        for (int idx = tid; idx < pk_total; idx += SV_THREADS) {
            const u64 g = base + (u64)idx;
            if (g < cap) { st_stream_u64(kout + g, stg_k[idx]); st_stream_d2(aout + g, stg_a[idx]); }
        }
        __syncthreads();          // staging (and s_base) are free again
        pk_valid = false;
    };

    const u32 tile0 = first_tile_of_block<!PRE>();
    if constexpr (TWO) {
        if (tid < SV_PIECES2_WORDS) s_desc[0][tid] = (reinterpret_cast<const u64*>(desc) + (size_t)tile0 * SV_PIECES2_WORDS)[tid];
        __syncthreads();
        if (tid == 0) issue_loads2(s_desc[0], 0, La0);
        __syncthreads();      // the piece table of the first tile is visible
    } else {
        if (tid < 8) s_desc[0][tid] = reinterpret_cast<const u64*>(desc + tile0)[tid];
        __syncthreads();
        issue_loads(pieces_of(s_desc[0]), La0);
    }
    int par = 0;
    for (u32 tile = tile0; tile < ntiles; tile += gridDim.x, par ^= 1) {
        const u32 next = tile + gridDim.x;
        double2* La = par ? La1 : La0;     // this tile's amplitudes, by landing index
        u64 dnext = 0;
        if constexpr (TWO) { if (tid < SV_PIECES2_WORDS && next < ntiles) dnext = (reinterpret_cast<const u64*>(desc) + (size_t)next * SV_PIECES2_WORDS)[tid]; }
        else { if (tid < 8 && next < ntiles) dnext = reinterpret_cast<const u64*>(desc + next)[tid]; }
        Pieces3 pc;
        if constexpr (!TWO) pc = pieces_of(s_desc[par]); else { pc.cnt = s_pcum[par][DP_MAXPIECES]; pc.oneblock = false; pc.l0 = 0; }
        const int cnt = pc.cnt;
        int nA, nL;
        {   // pick up this thread's landed elements, apply a pending truncation, partition the LIVE ones into A* | B*
            mbar_wait(&s_bar, bar_phase);      // the tile has landed
            bar_phase ^= 1u;
            Landing3 ld;
            if constexpr (!TWO) ld = landing_of(pc);
            int pcs[TWO ? DP_MAXPIECES : 1];          // TWO: first load-order index of pieces 1 .. 7
            if constexpr (TWO) {
#pragma unroll
                for (int i = 1; i < DP_MAXPIECES; ++i) pcs[i] = s_pcum[par][i];
            }
            u64 lk[BP_VT]; double2 la[BP_VT];
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const int e = tid + r * SV_THREADS;
                lk[r] = 0; la[r] = make_double2(0.0, 0.0);
                if (e < cnt) {
                    if constexpr (TWO) {
                        int q = 0;
#pragma unroll
                        for (int i = 1; i < DP_MAXPIECES; ++i) q += (e >= pcs[i]) ? 1 : 0;
                        const int sl = e + s_pko[par][q];
                        SV_CHK(sl >= 0 && sl < BP_TILE + LKX);
                        lk[r] = Lk[sl];
                    } else lk[r] = Lk[landing_key_slot(pc, ld, e)];
                    la[r] = La[e];
                }
            }
            if (pd.active) {   // (survivors are rescaled in place; what the cut drops is not given a slot below)
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    if (tid + r * SV_THREADS < cnt) {
                        if (pend_keep(pd, lk[r], la[r])) {
                            la[r].x = __dmul_rn(la[r].x, pd.scale); la[r].y = __dmul_rn(la[r].y, pd.scale);
                            La[tid + r * SV_THREADS] = la[r];
                        } else { la[r].x = 0.0; la[r].y = 0.0; }
                    }
                }
            }
            if constexpr (TWO) {
                // the live entries by class (bH, bL), each class in load order = ascending rest; keys -> (high, mid, low, bH, bL):
                // with the two bits at the bottom a plain comparison orders both merges (equal rest: bL = 0, bH = 0 first)
                u32 bal[4][BP_VT];
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    const bool live = (tid + r * SV_THREADS < cnt) && !(la[r].x == 0.0 && la[r].y == 0.0);
                    const u32 bl = __ballot_sync(0xffffffffu, live);
                    const u32 bh = __ballot_sync(0xffffffffu, (lk[r] & bit) != 0), b2 = __ballot_sync(0xffffffffu, (lk[r] & bit2) != 0);
                    bal[0][r] = bl & ~bh & ~b2; bal[1][r] = bl & ~bh & b2; bal[2][r] = bl & bh & ~b2; bal[3][r] = bl & bh & b2;
                    const u32 mine = lane == 0 ? bal[0][r] : (lane == 1 ? bal[1][r] : (lane == 2 ? bal[2][r] : bal[3][r]));
                    if (lane < 4) wc4[lane][r][warp] = __popc(mine);
                }
                __syncthreads();
                if (warp < 4) {   // lane = r * 8 + w: exclusive scan of the 32 counts of class `warp` in load order
                    int* wv = &wc4[warp][0][0];
                    const int c = wv[lane];
                    int inc = c;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                    wv[lane] = inc - c;
                    if (lane == 31) s_n4[warp] = inc;
                }
                __syncthreads();
                const int n00 = s_n4[0], n01 = s_n4[1], n10 = s_n4[2];
                nA = n00 + n01; nL = nA + n10 + s_n4[3];
                const int cb[4] = {0, n00, nA, nA + n10};
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    int slot = -1;
#pragma unroll
                    for (int c = 0; c < 4; ++c)
                        if ((bal[c][r] >> lane) & 1u) slot = cb[c] + wc4[c][r][warp] + __popc(bal[c][r] & lt);
                    SV_CHK(slot < nL);
                    if (slot >= 0) {
                        const u64 k = lk[r];
                        sk[DK(slot)] = (k & himask) | ((k & midmask) << 1) | ((k & lowmask2) << 2) | ((k & bit) ? 2ull : 0ull) | ((k & bit2) ? 1ull : 0ull);
                        si[slot] = (unsigned short)(tid + r * SV_THREADS);
                    }
                }
            } else if (!maybe_dead && (!mv || pc.oneblock)) {   // load order = A* | B* already and nothing to squeeze out
                nA = mv ? pc.l0 : cnt; nL = cnt;
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    const int e = tid + r * SV_THREADS;
                    if (e < cnt) { sk[DK(e)] = lk[r] & ~bit; si[e] = (unsigned short)e; }
                }
            } else {
                u32 balA[BP_VT], balB[BP_VT];
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    const bool live = (tid + r * SV_THREADS < cnt) && !(la[r].x == 0.0 && la[r].y == 0.0);
                    const bool isB = live && (lk[r] & bit);
                    balA[r] = __ballot_sync(0xffffffffu, live && !isB);
                    balB[r] = __ballot_sync(0xffffffffu, isB);
                    if (lane == 0) { wcA[r][warp] = __popc(balA[r]); wcB[r][warp] = __popc(balB[r]); }
                }
                __syncthreads();
                if (warp < 2) {   // lane = r * 8 + warp: exclusive scans of the 32 counts in load order (A: warp 0, B: warp 1)
                    int* w = warp == 0 ? &wcA[0][0] : &wcB[0][0];
                    const int c = w[lane];
                    int inc = c;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                    w[lane] = inc - c;
                    if (lane == 31) { if (warp == 0) s_nA = inc; else s_nB = inc; }
                }
                __syncthreads();
                nA = s_nA; nL = nA + s_nB;
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    int slot = -1;
                    if ((balA[r] >> lane) & 1u) slot = wcA[r][warp] + __popc(balA[r] & lt);
                    else if ((balB[r] >> lane) & 1u) slot = nA + wcB[r][warp] + __popc(balB[r] & lt);
                    SV_CHK(slot < nL);
                    if (slot >= 0) { sk[DK(slot)] = lk[r] & ~bit; si[slot] = (unsigned short)(tid + r * SV_THREADS); }
                }
            }
        }
        if (tid < (TWO ? SV_PIECES2_WORDS : 8) && next < ntiles) s_desc[par ^ 1][tid] = dnext;
        __syncthreads();
        if constexpr (TWO) { if (next < ntiles && tid == 0) issue_loads2(s_desc[par ^ 1], par ^ 1, par ? La0 : La1); }
        else { if (next < ntiles) issue_loads(pieces_of(s_desc[par ^ 1]), par ? La0 : La1); }

        // ---- TWO, level 1: inside either bH class, merge its bL = 0 and bL = 1 entries by the rest of the key (two merges
        // side by side over the output positions [0, nA) and [nA, nL)); bL goes to bit 0 ----
        if constexpr (TWO) {
            const int n00 = s_n4[0], n10 = s_n4[2];
            const int d0 = min(tid * BP_VT, nL);
            int seg = (d0 >= nA) ? 1 : 0;
            int ob = seg ? nA : 0;          // first entry of this thread's pair of classes
            int na = seg ? n10 : n00, nb = seg ? (nL - nA - n10) : (nA - n00);
            const int dg = d0 - (seg ? nA : 0);
            int i, j;
            {
                int lo = max(0, dg - nb), hi = min(dg, na);
                while (lo < hi) {   // bL = 0 first on ties
                    const int mid = (lo + hi) >> 1;
                    if (sk[DK(ob + mid)] <= sk[DK(ob + na + dg - 1 - mid)]) lo = mid + 1; else hi = mid;
                }
                i = lo; j = dg - lo;
            }
            u64 ka = (i < na) ? sk[DK(ob + i)] : ~0ull, kb = (j < nb) ? sk[DK(ob + na + j)] : ~0ull;
            u64 mk[BP_VT]; unsigned short mi[BP_VT];
#pragma unroll
            for (int v = 0; v < BP_VT; ++v) {
                mk[v] = 0; mi[v] = 0;
                if (d0 + v < nL) {
                    if (seg == 0 && d0 + v == nA) {   // this thread's outputs run over into the bH = 1 merge: it starts there
                        seg = 1; ob = nA; na = n10; nb = nL - nA - n10; i = 0; j = 0;
                        ka = (0 < na) ? sk[DK(ob)] : ~0ull; kb = (0 < nb) ? sk[DK(ob + na)] : ~0ull;
                    }
                    const bool takeA = ka <= kb;
                    mk[v] = takeA ? ka : kb;
                    mi[v] = si[takeA ? ob + i : ob + na + j];
                    if (takeA) { ++i; ka = (i < na) ? sk[DK(ob + i)] : ~0ull; } else { ++j; kb = (j < nb) ? sk[DK(ob + na + j)] : ~0ull; }
                }
            }
            __syncthreads();   // every read of the partitioned tile is done
#pragma unroll
            for (int v = 0; v < BP_VT; ++v)
                if (d0 + v < nL) { sk[DK(d0 + v)] = mk[v]; si[d0 + v] = mi[v]; }
            __syncthreads();
        }

        // ---- phase 1: bring the tile into its new order (moved bit at the LSB) ----
        if (mv) {
            const int nB = nL - nA;
            const int diag = min(tid * BP_VT, nL);
            int i, j;
            {
                int lo = max(0, diag - nB), hi = min(diag, nA);
                while (lo < hi) {   // A first on ties
                    const int mid = (lo + hi) >> 1;
                    if (sk[DK(mid)] <= sk[DK(nA + diag - 1 - mid)]) lo = mid + 1; else hi = mid;
                }
                i = lo; j = diag - lo;
            }
            SV_CHK(i >= 0 && i <= nA && j >= 0 && j <= nB);
            const int endpos = min(diag + BP_VT, nL);
            u64 ka = (i < nA) ? sk[DK(i)] : ~0ull, kb = (j < nB) ? sk[DK(nA + j)] : ~0ull;
            u64 mk[BP_VT]; unsigned short mi[BP_VT];
#pragma unroll
            for (int v = 0; v < BP_VT; ++v) {
                mk[v] = 0; mi[v] = 0;
                if (diag + v < endpos) {
                    const bool takeA = ka <= kb;
                    const u64 k = takeA ? ka : kb;
                    mi[v] = si[takeA ? i : nA + j];
                    mk[v] = TWO ? k : ((k & himask) | ((k & lowmask) << 1) | (takeA ? 0ull : 1ull));
                    if (takeA) { ++i; ka = (i < nA) ? sk[DK(i)] : ~0ull; } else { ++j; kb = (j < nB) ? sk[DK(nA + j)] : ~0ull; }
                }
            }
            // The tuples are found here, from the merged keys in registers: a thread's outputs are consecutive, its
            // predecessor's last key comes by shuffle (across warps through shared memory, behind the barrier the
            // merge needs anyway).  The tile's tuple count -- hence, two calls, its output count -- is known two
            // barriers earlier than with a pass of its own over the merged tile, and is published at once.
            u64 mylast = 0ull;
#pragma unroll
            for (int v = 0; v < BP_VT; ++v) if (diag + v < endpos) mylast = mk[v];
            if (lane == 31) s_last[warp] = mylast;          // (a thread without elements sits behind the tile's end: never read)
            __syncthreads();   // every read of the partitioned tile is done
            u64 prev = __shfl_up_sync(0xffffffffu, mylast, 1);
            if (lane == 0 && warp > 0) prev = s_last[warp - 1];
            u32 om = 0;        // bit v: merged element diag + v opens a tuple
#pragma unroll
            for (int v = 0; v < BP_VT; ++v) {
                if (diag + v < endpos) {
                    const u64 before = v == 0 ? prev : mk[v - 1];
                    if ((diag + v == 0) || (before >> MA) != (mk[v] >> MA)) om |= 1u << v;
                    sk[DK(diag + v)] = mk[v]; si[diag + v] = mi[v];
                }
            }
            int cinc = __popc(om);
            const int cmine = cinc;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, cinc, d); if (lane >= d) cinc += t; }
            if (lane == 31) wcA[0][warp] = cinc;
            __syncthreads();   // merged tile and the warps' tuple counts visible
            int tbefore = 0, tall = 0;
#pragma unroll
            for (int w = 0; w < BP_WARPS; ++w) { const int c = wcA[0][w]; tall += c; if (w < warp) tbefore += c; }
            if (!PRE && tid == 0) lookback_publish(status, gstat, tile, ntiles, (u64)tall << MA);   // known before any arithmetic
            int tix = tbefore + cinc - cmine;
#pragma unroll
            for (int v = 0; v < BP_VT; ++v)
                if ((om >> v) & 1u) tst[tix++] = (unsigned short)(diag + v);
            if (tid == 0) { tst[tall] = (unsigned short)nL; s_nt = tall; }
        } else {
        // ---- phase 2 (no move): tuples (elements taken strided: conflict-free reads; counts scanned in element order) ----
            u32 bs[BP_VT];
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const int e = tid + r * SV_THREADS;
                const bool opens = (e < nL) && (e == 0 || (sk[DK(e - 1)] >> MA) != (sk[DK(e)] >> MA));
                bs[r] = __ballot_sync(0xffffffffu, opens);
                if (lane == 0) wcA[r][warp] = __popc(bs[r]);
            }
            __syncthreads();
            if (warp == 0) {
                int* w = &wcA[0][0];
                const int c = w[lane];
                int inc = c;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                w[lane] = inc - c;
                if (lane == 31) s_nt = inc;
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < BP_VT; ++r)
                if ((bs[r] >> lane) & 1u) tst[wcA[r][warp] + __popc(bs[r] & lt)] = (unsigned short)(tid + r * SV_THREADS);
            if (tid == 0) tst[s_nt] = (unsigned short)nL;
            if (!PRE && tid == 0) lookback_publish(status, gstat, tile, ntiles, (u64)s_nt << MA);   // known before any arithmetic
        }
        __syncthreads();              // tuple table complete
        const int NT = s_nt;
        SV_CHK(NT >= 0 && NT <= nL && nL <= BP_TILE);
        const int NC = NT << MA;      // candidates of the tile
        if (PRE && pk_valid) flush_parked();   // (the look-back of the previous tile has had the whole front end to resolve)

        // ---- back end: ONE THREAD PER TUPLE, all 2^MA rows in registers ----
        // A round takes 256 * TPR tuples; warp w the 32 * TPR consecutive ones from hw, lane l the tuples hw + u * 32 + l.
        u64 base = 0;
        bool have_base = false;     // !PRE: the look-back is resolved behind the first round's arithmetic
        int run = 0;                // PRE: survivors of the earlier rounds (uniform over the block)
        int wpar = 0;
        auto round_compute = [&](int hw, double (&accr)[TPR][NP], double (&acci)[TPR][NP], u64 (&kb)[TPR], bool (&valid)[TPR]) {
#pragma unroll
            for (int u = 0; u < TPR; ++u) {
                const int ti = hw + u * 32 + lane;
                valid[u] = ti < NT;
                kb[u] = 0;
#pragma unroll
                for (int r = 0; r < NP; ++r) { accr[u][r] = 0.0; acci[u][r] = 0.0; }
                if (valid[u]) {
                    const int e = tst[ti], nm = (int)tst[ti + 1] - e;
                    SV_CHK(nm >= 1 && nm <= NP && e + nm <= nL);
                    kb[u] = sk[DK(e)] & ~AM;
                    if (col_ident || nm <= 2) {          // members in stored order = ascending logical column (or the order cannot matter)
                        for (int j = 0; j < nm; ++j) {
                            const int x = (int)(sk[DK(e + j)] & AM);
                            SV_CHK(si[e + j] < cnt);
                            const double2 a = La[si[e + j]];
#pragma unroll
                            for (int r = 0; r < NP; ++r) {
                                const double2 uu = Us[r * NP + x];
                                cmul_acc(accr[u][r], acci[u][r], uu.x, uu.y, a.x, a.y);
                            }
                        }
                    } else {                              // ascending LOGICAL column index (D1)
                        u32 pk = 0;
                        for (int j = 0; j < nm; ++j) pk |= 1u << (int)(sk[DK(e + j)] & AM);
                        for (int t = 0; t < NP; ++t) {
                            const int x = (int)((colpack >> (4 * t)) & 15ull);
                            if ((pk >> x) & 1u) {
                                const double2 a = La[si[e + __popc(pk & ((1u << x) - 1u))]];
#pragma unroll
                                for (int r = 0; r < NP; ++r) {
                                    const double2 uu = Us[r * NP + x];
                                    cmul_acc(accr[u][r], acci[u][r], uu.x, uu.y, a.x, a.y);
                                }
                            }
                        }
                    }
                }
            }
        };
        if constexpr (!PRE) {
            // ---- two calls: every candidate is an output.  The 2^MA rows a thread holds are CONSECUTIVE outputs (64 bytes of
            // amplitudes, 32 of keys for MA = 2), the tuples of consecutive lanes follow one another, and a tile's first
            // output is a multiple of 2^MA: every thread stores its rows straight from registers with 256-bit stores, each a
            // whole 32-byte sector.  (Until round 2 every warp transposed its round through shared memory so that
            // consecutive lanes stored consecutive 16-byte entries: a third of the pass's shared-memory wavefronts.) ----
            for (int h = 0; h < NT; h += SV_THREADS * TPR) {
                const int hw = h + warp * (32 * TPR);
                double accr[TPR][NP], acci[TPR][NP]; u64 kb[TPR]; bool valid[TPR];
                round_compute(hw, accr, acci, kb, valid);
#pragma unroll
                for (int u = 0; u < TPR; ++u)
#pragma unroll
                    for (int r = 0; r < NP; ++r)
                        if (valid[u] && accr[u][r] == 0.0 && acci[u][r] == 0.0) ++n_dead;   // exact cancellation: a dead entry
                if (!have_base) {
                    if (tid < 32) {
                        const u64 ex = lookback_exclusive_2level<false>(status, gstat, tile, ntiles, (u64)NC);
                        if (tid == 0) {
                            s_base = ex;
                            if (tile == ntiles - 1) d_count[0] = ex + (u64)NC;
                        }
                    }
                    __syncthreads();
                    base = s_base; have_base = true;
                }
#pragma unroll
                for (int u = 0; u < TPR; ++u) {
                    if (!valid[u]) continue;
                    const u64 g0 = base + ((u64)(hw + u * 32 + lane) << MA);
                    if (g0 + (u64)NP <= cap) {
#pragma unroll
                        for (int r = 0; r < NP; r += 4)
                            st_stream_u64x4(kout + g0 + r, kb[u] | (u64)r, kb[u] | (u64)(r + 1), kb[u] | (u64)(r + 2), kb[u] | (u64)(r + 3));
#pragma unroll
                        for (int r = 0; r < NP; r += 2)
                            st_stream_d2x2(aout + g0 + r, accr[u][r], acci[u][r], accr[u][r + 1], acci[u][r + 1]);
                    } else {
#pragma unroll
                        for (int r = 0; r < NP; ++r)
                            if (g0 + (u64)r < cap) { st_stream_u64(kout + g0 + r, kb[u] | (u64)r); st_stream_d2(aout + g0 + r, make_double2(accr[u][r], acci[u][r])); }
                    }
                }
            }
            if (!have_base) {   // (a tile without a live term still takes part in the chain)
                if (tid < 32) {
                    const u64 ex = lookback_exclusive_2level<false>(status, gstat, tile, ntiles, (u64)NC);
                    if (tid == 0 && tile == ntiles - 1) d_count[0] = ex + (u64)NC;
                }
            }
        } else {
            // ---- fused apply + truncate: compute once, keep what reaches the floor, rank, stage in output order ----
            auto rounds = [&](auto direct_tag) {
                constexpr bool DIRECT = decltype(direct_tag)::value;
                run = 0;
                for (int h = 0; h < NT; h += SV_THREADS * TPR, wpar ^= 1) {
                    const int hw = h + warp * (32 * TPR);
                    double accr[TPR][NP], acci[TPR][NP]; u64 kb[TPR]; bool valid[TPR];
                    round_compute(hw, accr, acci, kb, valid);
                    u32 mask[TPR]; int ex[TPR];
                    int wsum = 0;
#pragma unroll
                    for (int u = 0; u < TPR; ++u) {
                        u32 m = 0;
#pragma unroll
                        for (int r = 0; r < NP; ++r) {
                            if (valid[u] && !(accr[u][r] == 0.0 && acci[u][r] == 0.0)) {   // (an exact cancellation is simply not written)
                                const double pr = prob_of(make_double2(accr[u][r], acci[u][r]));
                                if ((u64)__double_as_longlong(pr) >= Pf) m |= 1u << r;
                                else if (!DIRECT) { dmass = __dadd_rn(dmass, pr); ++dcnt; }
                            }
                        }
                        mask[u] = m;
                        const int c = __popc(m);
                        int inc = c;
#pragma unroll
                        for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
                        ex[u] = wsum + inc - c;
                        wsum += __shfl_sync(0xffffffffu, inc, 31);
                    }
                    if (lane == 0) wtot[wpar][warp] = wsum;
                    __syncthreads();
                    int woff = 0, rtot = 0;
#pragma unroll
                    for (int w = 0; w < BP_WARPS; ++w) { const int c = wtot[wpar][w]; rtot += c; if (w < warp) woff += c; }
#pragma unroll
                    for (int u = 0; u < TPR; ++u) {
                        int s = run + woff + ex[u];
#pragma unroll
                        for (int r = 0; r < NP; ++r) {
                            if ((mask[u] >> r) & 1u) {
                                if (DIRECT) {
                                    const u64 g = base + (u64)s;
                                    if (g < cap) { st_stream_u64(kout + g, kb[u] | (u64)r); st_stream_d2(aout + g, make_double2(accr[u][r], acci[u][r])); }
                                } else if (s < DP_STAGE) { stg_k[s] = kb[u] | (u64)r; stg_a[s] = make_double2(accr[u][r], acci[u][r]); }
                                ++s;
                            }
                        }
                    }
                    run += rtot;
                }
            };
            rounds(std::false_type{});
            const int total = run;
            SV_CHK(total >= 0 && total <= NC);
            if (tid == 0) lookback_publish(status, gstat, tile, ntiles, (u64)total);
            if (total <= DP_STAGE) {      // parked: stored after the next tile's front end
                pk_valid = true; pk_tile = tile; pk_total = total;
            } else {                      // more survivors than the staging buffer holds: second evaluation, direct stores
                if (tid < 32) {
                    const u64 ex = lookback_exclusive_2level<false>(status, gstat, tile, ntiles, (u64)total);
                    if (tid == 0) {
                        s_base = ex;
                        if (tile == ntiles - 1) d_count[0] = ex + (u64)total;
                    }
                }
                __syncthreads();
                base = s_base;
                rounds(std::true_type{});
            }
        }
        __syncthreads();   // the tile and the tuple table are reused by the next tile
    }
    if (PRE && pk_valid) flush_parked();
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) n_dead += __shfl_xor_sync(0xffffffffu, n_dead, d);
    if (lane == 0 && n_dead) atomicAdd(reinterpret_cast<unsigned long long*>(&d_count[1]), (unsigned long long)n_dead);
    if (PRE) {   // block totals of what was left out, summed in a fixed order (see sv_pair.cu)
        __shared__ double s_pm[BP_WARPS];
        __shared__ u32 s_pc[BP_WARPS];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            dmass = __dadd_rn(dmass, __shfl_xor_sync(0xffffffffu, dmass, d));
            dcnt += __shfl_xor_sync(0xffffffffu, dcnt, d);
        }
        if (lane == 0) { s_pm[warp] = dmass; s_pc[warp] = dcnt; }
        __syncthreads();
        if (tid == 0) {
            double m = 0.0; u64 c = 0;
            for (int w = 0; w < BP_WARPS; ++w) { m = __dadd_rn(m, s_pm[w]); c += s_pc[w]; }
            pre_mass[blockIdx.x] = m; pre_cnt[blockIdx.x] = c;
        }
    }
}

template <int MA, bool PRE, bool TWO>
static u32 launch_densepass(const u64* kin, const double2* ain, u64* kout, double2* aout, int p, const GateTab* tab,
                            const PendPred& pend, TileDesc* desc, u64* status, u64* d_count, u64 cap, u32 ntiles, cudaStream_t st,
                            const PreCut* pre, double* pre_mass, u64* pre_cnt, int maybe_dead, int p2) {
    const size_t smem = (size_t)2 * BP_TILE * 24 + (TWO ? 128 : 64) + (size_t)(BP_TILE + 8) * 2 + (size_t)BP_TILE * 2 +
                        (PRE ? (size_t)DP_STAGE * 24 : 0);   // (two calls: the outputs are stored straight from registers)
    static int per_sm[SV_MAX_DEV];
    return sv_launch_persistent(densepass_kernel<MA, PRE, TWO>, per_sm, smem, ntiles, st, kin, ain, kout, aout, p, tab, pend,
                                (const TileDesc*)desc, status, d_count, cap, ntiles, pre, pre_mass, pre_cnt, maybe_dead, p2);
}

// Dispatch for svk_grouppass (sv_group.cu): the final pass of a dense gate.  Returns the grid size.
u32 svk_densepass_launch(int ma, bool use_pre, const u64* kin, const double2* ain, u64* kout, double2* aout, int p, const GateTab* tab,
                         const PendPred& pend, TileDesc* desc, u64* status, u64* d_count, u64 cap, u32 ntiles, cudaStream_t st,
                         const PreCut* pre, double* pre_mass, u64* pre_cnt, int maybe_dead, int p2) {
#define SV_DP(MA_, PRE_) launch_densepass<MA_, PRE_, true>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st, pre, pre_mass, pre_cnt, maybe_dead, p2)
    if (p2 >= 0) {   // two bits moved by this pass (desc: the piece table of make_pieces2); two calls only (sv_api.cu)
        if (use_pre) return 0;
        switch (ma) { case 2: return SV_DP(2, false); case 3: return SV_DP(3, false); case 4: return SV_DP(4, false); default: return 0; }
    }
#undef SV_DP
#define SV_DP(MA_, PRE_) launch_densepass<MA_, PRE_, false>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st, pre, pre_mass, pre_cnt, maybe_dead, -1)
    if (use_pre) {
        switch (ma) { case 2: return SV_DP(2, true); case 3: return SV_DP(3, true); case 4: return SV_DP(4, true); default: return 0; }
    }
    switch (ma) { case 2: return SV_DP(2, false); case 3: return SV_DP(3, false); case 4: return SV_DP(4, false); default: return 0; }
#undef SV_DP
}

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
// The pass is bound by the shared-memory pipe, not by HBM (profiles/r1_b_pipeline.md), so the
// data flow keeps shared-memory traffic low: ONLY KEYS are partitioned, searched and merged;
// an amplitude lands once (cp.async, double buffered) and is read once, by index, where it is
// needed.
//
//   land      the tile's (up to three) contiguous pieces arrive through cp.async one tile ahead;
//   prepare   every thread files the keys it requested into A* | B* (bit p cleared) together with
//             their landing slot;
//   split     every thread finds where its VT consecutive OUTPUT positions start in A* and B*
//             (merge path: one binary search per thread, not per term);
//   merge     VT sequential merge steps per thread over keys.  Partners (the
//             terms that differ only in the gate's qubit) meet as neighbours;
//   write     MODE 0 / 2 (position preserving, see FIXED below): output keys and source slots are
//             staged by output position; the copy-out gathers each amplitude from the landing
//             buffer, applies a pending truncation (dropped -> dead entry 0+0i, survivors scaled)
//             and the gate's phase, and stores coalesced.
//             MODE 1 (general 2x2 blocks): the tuple mat-vec runs in the merge,
//             exact zeros are dropped, block scan + two-level look-back give the
//             offsets, outputs are staged and stored coalesced: sorted, unique keys by construction.
#include "sv_tile.cuh"
#include "sv_launch.cuh"

// MODE 0: pure move.  MODE 1: gate with one active bit (2x2 mat-vec per tuple).  MODE 2 (FIXED only):
// the same for MONOMIAL 2x2 blocks: every entry maps to one entry (its bit kept or flipped, times a
// phase), so the pass is a move whose partners may trade places -- no tuple arithmetic.
// FIXED: position-preserving variant for passes that map every stored entry to exactly one stored
// entry (pure moves, monomial blocks).  Terms dropped by a pending truncation are carried as DEAD
// entries (amplitude 0+0i) instead of being squeezed out, so the position of every output is known
// from the tile descriptor alone: no scan, no look-back.
// Staged outputs are written by threads that each own a few CONSECUTIVE output positions: without a
// skew all lanes of a warp would hit the same banks (stride 4..8 entries).  The column (entry index
// within a 128-byte row: 16 keys / 8 amplitudes) is XORed with the row index, which spreads such
// writes over the banks and keeps the copy-out reads of consecutive entries inside one row.
#define BP_SWK(x) ((x) ^ (((x) >> 4) & 15))
#define BP_SWA(x) ((x) ^ (((x) >> 3) & 7))
#ifndef BP_GEN2_CTAS
#define BP_GEN2_CTAS 4                         // resident blocks per SM of the general one-bit pass, two calls.  4 (64 registers, no second
#endif                                         // key array, hence no parking): its tiles hold > 1024 outputs and could not park anyway; the
                                               // fourth block hides their look-back wait better: H apply 5.07 -> 4.83 ms
#ifndef BP_GENP_CTAS
#define BP_GENP_CTAS 3                         // the same, fused call (3: tiles park, see BP_PARK_EXTRA)
#endif
#ifndef BP_GEN_CTAS
#define BP_GEN_CTAS 3                          // resident blocks per SM of the general one-bit pass (0: BP_CTAS)
#endif
#define BP_WKN BP_TILE                         // entries of the key / slot work arrays
#define BP_ROUND BP_TILE                       // outputs staged per round when amplitudes are staged too
#ifndef BP_PARK_EXTRA
#define BP_PARK_EXTRA 256                      // general one-bit pass of the FUSED call: a staging round holds this many outputs more than a tile has
#endif                                         // inputs, so that the fused call's tiles (~1.02 outputs per input) fit one round and park
// PRE (MODE 1 only; fused apply + truncate, sv_presample.cu): outputs whose probability pattern is below
// pre->P_floor are not written; every block leaves the mass and the number of what it left out in
// pre_mass / pre_cnt[blockIdx.x] (tiles are taken in a fixed order, so these sums are the same every run).
template <int MODE, bool FIXED, bool PRE>
__global__ void __launch_bounds__(SV_THREADS, (MODE == 1 && BP_GEN_CTAS) ? (PRE ? BP_GENP_CTAS : BP_GEN2_CTAS) : BP_CTAS) bitpass_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                                u64* __restrict__ kout, double2* __restrict__ aout, int p,
                                                                const GateTab* __restrict__ gtab, PendPred pd,
                                                                const TileDesc* __restrict__ desc, u64* status,
                                                                u64* d_count, u64 cap, u32 ntiles, const PreCut* __restrict__ pre,
                                                                double* __restrict__ pre_mass, u64* __restrict__ pre_cnt) {
    constexpr bool PAIR = (MODE == 1);
    constexpr bool PERM = (MODE == 2);
    constexpr int STG = BP_TILE + ((!FIXED && MODE == 1 && PRE && BP_GENP_CTAS < 4) ? BP_PARK_EXTRA : 0);   // entries of the amplitude buffers and key work arrays
    constexpr int ROUND = STG;                                                   // outputs staged per round
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* La0 = reinterpret_cast<double2*>(smem_raw);       // landing amplitudes, double buffered
    double2* La1 = La0 + STG;
    u64* Lk = reinterpret_cast<u64*>(La1 + STG);           // landing keys (consumed by prepare)
    u64* Wk0 = Lk + BP_TILE + 8;                               // A* | B* keys with bit p cleared; later the staged output keys
    unsigned short* Wi = reinterpret_cast<unsigned short*>(Wk0 + STG);   // their landing slots; later the staged source slots
    // PARK (general one-bit gate): a second key array, used in turns with the first, so that a tile whose outputs fit
    // one round leaves them parked in shared memory (keys there, amplitudes in the tile's landing buffer), publishes
    // its total at once and goes on with the block's next tile; its look-back is resolved after that tile's prepare
    // step: the chain of L2 round trips (tile totals -> group total -> reader) has run
    // behind that work instead of holding the whole block at a barrier.
    constexpr bool PARK = !FIXED && MODE == 1 && (PRE ? BP_GENP_CTAS < 4 : BP_GEN2_CTAS < 4);   // (the compacting move keeps 4 resident blocks: no room for the array)
    u64* Wk1 = PARK ? reinterpret_cast<u64*>(Wi + STG) : Wk0;
    bool pk_valid = false;      // uniform over the block
    u32 pk_tile = 0; int pk_total = 0;
    u64* pk_keys = Wk0; double2* pk_amps = La0;
    __shared__ int red[BP_WARPS + 2];
    __shared__ int wc[BP_VT][BP_WARPS];
    __shared__ int s_nA;
    __shared__ u64 s_desc[2][8];
    __shared__ u64 s_base;
    __shared__ __align__(8) u64 s_bar;   // mbarrier of the landing bulk copies (one batch in flight at a time)
    __shared__ double2 sU[64];      // [cx][xr][xc], ma = 1: up to 8 control patterns x 4
    __shared__ int s_cpos[SV_MAX_M], s_mc;
    __shared__ int s_sw[8], s_unit; // PERM: block cx swaps the bit; every nonzero entry is exactly 1
    __shared__ int s_ctrl_only;     // PERM: only the all-ones control pattern swaps (CNOT, Toffoli, C3X)
    __shared__ u64 s_cmask;         // PERM: the control bits (new layout)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (PAIR || PERM) {
        if (tid < 64) sU[tid] = gtab->U[tid];
        if (tid < SV_MAX_M) s_cpos[tid] = gtab->ctrl_pos[tid];
        if (tid == 0) s_mc = gtab->mc;
        if (PERM && tid == 0) {
            int unit = 1;
            for (int cx = 0; cx < 8; ++cx) {
                const double2* u = &gtab->U[cx << 2];
                const int sw = (u[0].x == 0.0 && u[0].y == 0.0) ? 1 : 0;
                s_sw[cx] = sw;
                const double2 x = sw ? u[1] : u[0], y = sw ? u[2] : u[3];
                if (cx < (1 << gtab->mc) && !(x.x == 1.0 && x.y == 0.0 && y.x == 1.0 && y.y == 0.0)) unit = 0;
            }
            s_unit = unit;
            const int full = (1 << gtab->mc) - 1;
            int co = 1;
            u64 cm = 0;
            for (int cx = 0; cx <= full; ++cx) if (s_sw[cx] != (cx == full ? 1 : 0)) co = 0;
            for (int q = 0; q < gtab->mc; ++q) cm |= 1ull << gtab->ctrl_pos[q];
            s_ctrl_only = co; s_cmask = cm;
        }
    }
    const u64 bit = 1ull << p;
    const u64 himask = (p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    const u64 Pf = PRE ? pre->P_floor : 0ull;
    double dmass = 0.0;     // PRE: mass and number of the outputs this thread left out
    u32 dcnt = 0;
    u64* gstat = status + ntiles;                       // group statuses follow the tile statuses
    // Persistent blocks (the grid is sized to be fully resident): tile t is taken by block t mod gridDim.x,
    // so a block only ever waits on tiles that resident blocks have taken already.  While a tile is
    // merged and written, the block's NEXT tile is already on its way from HBM (cp.async, one thread per
    // element): every block keeps a full tile of loads in flight.  Each thread later files exactly the
    // keys it requested.  Tile descriptors travel one iteration ahead (s_desc).
    // The tile lands by bulk copies (TMA): one thread arms the barrier and issues up to six copies (sv_tile.cuh).
    auto issue_loads = [&](const Pieces3& q, double2* La) {
        if (tid == 0) land_tile_bulk(q, kin, ain, Lk, La, &s_bar);
    };
    if (tid == 0) { mbar_init(&s_bar, 1); fence_proxy_async_smem(); }
    u32 bar_phase = 0;
    const u32 tile0 = first_tile_of_block<(MODE == 1 && !FIXED && !PRE)>();
    if (tid < 8) s_desc[0][tid] = reinterpret_cast<const u64*>(desc + tile0)[tid];
    __syncthreads();
    issue_loads(pieces_of(s_desc[0]), La0);
    int par = 0;
    for (u32 tile = tile0; tile < ntiles; tile += gridDim.x, par ^= 1) {
        double2* La = par ? La1 : La0;          // this tile's amplitudes (by landing slot)
        double2* Lnext = par ? La0 : La1;
        u64* Wk = par ? Wk1 : Wk0;
        const u32 next = tile + gridDim.x;
        u64 dnext = 0;
        if (tid < 8 && next < ntiles) dnext = reinterpret_cast<const u64*>(desc + next)[tid];
        const Pieces3 pc = pieces_of(s_desc[par]);
        const int cnt = pc.cnt;
        int nA;
        {   // ---- prepare: keys only ----
            mbar_wait(&s_bar, bar_phase);      // the tile has landed
            bar_phase ^= 1u;
            const Landing3 ld = landing_of(pc);
            u64 lk[BP_VT];
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const int e = tid + r * SV_THREADS;
                lk[r] = (e < cnt) ? Lk[landing_key_slot(pc, ld, e)] : 0;
            }
            if (pc.oneblock) {   // piece 0 is all A, piece 1 all B: the load order is already A* | B*
                nA = pc.l0;
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    const int e = tid + r * SV_THREADS;
                    if (e < cnt) Wk[e] = lk[r] & ~bit;   // (the landing slot of entry e is e itself: Wi is not needed)
                }
            } else {             // stable partition by bit p (the load order is the stored order)
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
                        SV_CHK(slot >= 0 && slot < cnt);
                        Wk[slot] = lk[r] & ~bit; Wi[slot] = (unsigned short)e;
                    }
                }
            }
        }
        if (tid < 8 && next < ntiles) s_desc[par ^ 1][tid] = dnext;
        __syncthreads();       // A* | B* complete, every landed amplitude visible, landing keys consumed
        if (PARK && pk_valid) {   // the previous tile's parked outputs: resolve its look-back, store coalesced
            if (tid < 32) {
                const u64 ex = lookback_exclusive_2level<false>(status, gstat, pk_tile, ntiles, (u64)pk_total);
                if (tid == 0) {
                    s_base = ex;
                    if (pk_tile == ntiles - 1) *d_count = ex + (u64)pk_total;
                }
            }
            __syncthreads();
            const u64 base = s_base;
#pragma unroll
            for (int it = 0; it < ROUND / SV_THREADS; ++it) {
                const int idx = tid + it * SV_THREADS;
                const u64 g = base + (u64)idx;
                if (idx < pk_total && g < cap) { st_stream_u64(kout + g, pk_keys[BP_SWK(idx)]); st_stream_d2(aout + g, pk_amps[BP_SWA(idx)]); }
            }
            __syncthreads();   // the parked arrays are free again (the next loads land in pk_amps)
            pk_valid = false;
        }
        if (next < ntiles) issue_loads(pieces_of(s_desc[par ^ 1]), Lnext);
        const int nB = cnt - nA;
        const u64* WkB = Wk + nA;
        const unsigned short* WiB = Wi + nA;

        // ---- merge-path split of this thread's first output position ----
        const int diag = min(tid * BP_VT, cnt);
        int i, j;
        {
            int lo = max(0, diag - nB), hi = min(diag, nA);
            while (lo < hi) {   // A first on ties
                const int mid = (lo + hi) >> 1;
                if (Wk[mid] <= WkB[diag - 1 - mid]) lo = mid + 1; else hi = mid;
            }
            i = lo; j = diag - lo;
        }
        SV_CHK(i >= 0 && i <= nA && j >= 0 && j <= nB);
        const int endpos = min(diag + BP_VT, cnt);
        int pos = diag;
        // keys with bit p cleared never equal ~0: safe sentinels for an exhausted side
        u64 ka = (i < nA) ? Wk[i] : ~0ull, kb = (j < nB) ? WkB[j] : ~0ull;
        if (FIXED) {
            // ---- keys only: output key, source slot and output position of VT merged terms ----
            u64 okey[BP_VT]; int osrc[BP_VT], opos[BP_VT];
            u64 lastA = (PERM && i > 0) ? Wk[i - 1] : ~0ull;   // PERM: a B term's partner is the A term merged just before it
            const bool ctrl_only = PERM && s_ctrl_only;
            const u64 cmask = PERM ? s_cmask : 0ull;
            const int mc_m = PERM ? s_mc : 0;
#pragma unroll
            for (int v = 0; v < BP_VT; ++v) {
                okey[v] = 0; osrc[v] = 0; opos[v] = -1;
                if (pos < endpos) {
                    const bool takeA = ka <= kb;
                    const u64 k = takeA ? ka : kb;
                    const u64 nk = (k & himask) | ((k & lowmask) << 1);     // new layout, LSB = 0
                    osrc[v] = pc.oneblock ? (takeA ? i : nA + j) : (takeA ? (int)Wi[i] : (int)WiB[j]);
                    int row = takeA ? 0 : 1, shift = 0;
                    if (PERM) {
                        const bool partner = takeA ? (kb == k) : (lastA == k);
                        int sw;
                        if (ctrl_only) sw = ((nk & cmask) == cmask) ? 1 : 0;
                        else {
                            int cx = 0;
                            for (int q = 0; q < mc_m; ++q) cx |= (int)((nk >> s_cpos[q]) & 1ull) << q;
                            sw = s_sw[cx];
                        }
                        osrc[v] |= (row << 15);                            // the term's ORIGINAL bit travels with its slot
                        if (partner && sw) shift = row ? -1 : 1;           // partners that swap rows trade places
                        row ^= sw;
                    }
                    okey[v] = nk | (u64)row;
                    opos[v] = pos + shift;
                    if (takeA) { ++i; lastA = k; ka = (i < nA) ? Wk[i] : ~0ull; } else { ++j; kb = (j < nB) ? WkB[j] : ~0ull; }
                    ++pos;
                }
            }
            __syncthreads();   // every read of A* | B* is done: stage by output position in the same arrays
#pragma unroll
            for (int v = 0; v < BP_VT; ++v)
                if (opos[v] >= 0) { SV_CHK(opos[v] < cnt && (osrc[v] & 0x7fff) < cnt); Wk[BP_SWK(opos[v])] = okey[v]; Wi[BP_SWK(opos[v])] = (unsigned short)osrc[v]; }
            __syncthreads();
            // ---- copy-out: gather the amplitude, apply a pending truncation and the phase, store coalesced ----
            const u64 base = s_desc[par][0] + s_desc[par][1] - s_desc[par][2];   // merged rank of the tile's first term
            const int mc = PERM ? s_mc : 0;
            const bool phase = PERM && !s_unit;
#pragma unroll
            for (int it = 0; it < BP_VT; ++it) {
                const int idx = tid + it * SV_THREADS;
                if (idx >= cnt) break;
                const u64 key = Wk[BP_SWK(idx)];
                const u32 code = Wi[BP_SWK(idx)];
                double2 a = La[code & 0x7fffu];
                const int row = (int)(key & 1ull);
                const int c = PERM ? (int)(code >> 15) : row;              // the bit the term had before the gate
                if (pd.active) {
                    const u64 old = (key & himask) | ((key >> 1) & lowmask) | (c ? bit : 0ull);   // the stored key it came from
                    if (pend_keep(pd, old, a)) { a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale); }
                    else { a.x = 0.0; a.y = 0.0; }
                }
                if (phase) {
                    int cx = 0;
                    for (int q = 0; q < mc; ++q) cx |= (int)((key >> s_cpos[q]) & 1ull) << q;
                    const double2 u = sU[(cx << 2) | (row << 1) | c];
                    const double pr = __dsub_rn(__dmul_rn(u.x, a.x), __dmul_rn(u.y, a.y));
                    const double pi = __dadd_rn(__dmul_rn(u.x, a.y), __dmul_rn(u.y, a.x));
                    a.x = __dadd_rn(0.0, pr); a.y = __dadd_rn(0.0, pi);
                }
                const u64 g = base + (u64)idx;
                if (g < cap) { st_stream_u64(kout + g, key); st_stream_d2(aout + g, a); }
            }
            __syncthreads();   // A* | B* and this landing buffer are reused
            continue;
        }

        // ---- compacting variants: amplitudes are read (by landing slot) in the merge ----
        auto amp_at = [&](int slot, u64 stored_key) {
            double2 a = La[slot];
            if (pd.active) {
                if (pend_keep(pd, stored_key, a)) { a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale); }
                else { a.x = 0.0; a.y = 0.0; }
            }
            return a;
        };
        u64 ok[BP_VT];
        double o0r[BP_VT], o0i[BP_VT], o1r[BP_VT], o1i[BP_VT];
        u32 fl = 0;     // two flag bits per step
        int nout = 0;
        if (PAIR && pos < endpos && j < nB && i > 0 && Wk[i - 1] == kb) {   // this B belongs to the previous thread's tuple
            ++j; ++pos;
            kb = (j < nB) ? WkB[j] : ~0ull;
        }
#pragma unroll
        for (int v = 0; v < BP_VT; ++v) {
            ok[v] = 0; o0r[v] = o0i[v] = o1r[v] = o1i[v] = 0.0;
            if (pos < endpos) {
                const bool takeA = ka <= kb;
                const u64 k = takeA ? ka : kb;
                const u64 nk = (k & himask) | ((k & lowmask) << 1);     // new layout, LSB = 0
                if (PAIR) {
                    // one code path for the common case (a term without its partner, from either run): the run only
                    // selects the landing slot and the column of U; a partner (rare in sparse states) adds its column
                    const int slot = pc.oneblock ? (takeA ? i : nA + j) : (takeA ? (int)Wi[i] : (int)WiB[j]);
                    const double2 a = amp_at(slot, takeA ? k : (k | bit));
                    const int c = takeA ? 0 : 1;
                    const bool has_partner = takeA && (kb == k);
                    if (takeA) { ++i; ka = (i < nA) ? Wk[i] : ~0ull; } else { ++j; kb = (j < nB) ? WkB[j] : ~0ull; }
                    ++pos;
                    int cx = 0;
                    const int mc = s_mc;
                    for (int q = 0; q < mc; ++q) cx |= (int)((nk >> s_cpos[q]) & 1ull) << q;
                    const double2* u = &sU[cx << 2];                    // u[xr * 2 + xc]
                    double r0 = 0.0, m0 = 0.0, r1 = 0.0, m1 = 0.0;
                    cmul_acc(r0, m0, u[c].x, u[c].y, a.x, a.y);
                    cmul_acc(r1, m1, u[2 + c].x, u[2 + c].y, a.x, a.y);
                    if (has_partner) {
                        const double2 pa = amp_at(pc.oneblock ? nA + j : (int)WiB[j], k | bit);
                        ++j; ++pos;
                        kb = (j < nB) ? WkB[j] : ~0ull;
                        cmul_acc(r0, m0, u[1].x, u[1].y, pa.x, pa.y);
                        cmul_acc(r1, m1, u[3].x, u[3].y, pa.x, pa.y);
                    }
                    u32 f0 = !(r0 == 0.0 && m0 == 0.0), f1 = !(r1 == 0.0 && m1 == 0.0);
                    if constexpr (PRE) {   // below the floor of the cut that follows: never written
                        const double p0 = prob_of(make_double2(r0, m0)), p1 = prob_of(make_double2(r1, m1));
                        if (f0 && (u64)__double_as_longlong(p0) < Pf) { f0 = 0; dmass = __dadd_rn(dmass, p0); ++dcnt; }
                        if (f1 && (u64)__double_as_longlong(p1) < Pf) { f1 = 0; dmass = __dadd_rn(dmass, p1); ++dcnt; }
                    }
                    ok[v] = nk; o0r[v] = r0; o0i[v] = m0; o1r[v] = r1; o1i[v] = m1;
                    fl |= (f0 | (f1 << 1)) << (2 * v);
                    nout += (int)(f0 + f1);
                } else {   // compacting move
                    const double2 a = takeA ? amp_at(pc.oneblock ? i : (int)Wi[i], k) : amp_at(pc.oneblock ? nA + j : (int)WiB[j], k | bit);
                    if (takeA) { ++i; ka = (i < nA) ? Wk[i] : ~0ull; } else { ++j; kb = (j < nB) ? WkB[j] : ~0ull; }
                    ++pos;
                    const u32 f0 = !(a.x == 0.0 && a.y == 0.0);
                    ok[v] = nk | (takeA ? 0ull : 1ull); o0r[v] = a.x; o0i[v] = a.y;
                    fl |= f0 << (2 * v);
                    nout += (int)f0;
                }
            }
        }
        int total;
        const int excl = block_excl_scan1(nout, red, &total);   // its barriers also retire every read of A* | B* and of the amplitudes
        // stage the outputs in output order (keys over A* | B*, amplitudes over this tile's landing buffer:
        // BP_ROUND outputs per round, a gate that doubles the tile is written in two rounds), store coalesced
        SV_CHK(total >= 0 && total <= 2 * BP_TILE && excl >= 0 && excl + nout <= total);
        const bool park = PARK && total <= ROUND;   // one round: its outputs wait in shared memory for the block's next tile
        if (tid == 0) lookback_publish(status, gstat, tile, ntiles, (u64)total);   // at once: the later tiles read it while this one stages
        for (int h0 = 0; h0 == 0 || h0 < total; h0 += ROUND) {
            if (h0 > 0) __syncthreads();
            {
                int off = excl - h0;
#pragma unroll
                for (int v = 0; v < BP_VT; ++v) {
                    const u32 f = (fl >> (2 * v)) & 3u;
                    if (f & 1u) {
                        if ((unsigned)off < (unsigned)ROUND) { Wk[BP_SWK(off)] = ok[v]; La[BP_SWA(off)] = make_double2(o0r[v], o0i[v]); }
                        ++off;
                    }
                    if (PAIR && (f & 2u)) {
                        if ((unsigned)off < (unsigned)ROUND) { Wk[BP_SWK(off)] = ok[v] | 1ull; La[BP_SWA(off)] = make_double2(o1r[v], o1i[v]); }
                        ++off;
                    }
                }
            }
            if (park) {
                pk_valid = true; pk_tile = tile; pk_total = total; pk_keys = Wk; pk_amps = La;
                break;
            }
            if (h0 == 0 && tid < 32) {
                const u64 ex = lookback_exclusive_2level<false>(status, gstat, tile, ntiles, (u64)total);
                if (tid == 0) {
                    s_base = ex;
                    if (tile == ntiles - 1) *d_count = ex + (u64)total;
                }
            }
            __syncthreads();
            const u64 base = s_base + (u64)h0;
            const int m = min(total - h0, ROUND);
#pragma unroll
            for (int it = 0; it < ROUND / SV_THREADS; ++it) {
                const int idx = tid + it * SV_THREADS;
                const u64 g = base + (u64)idx;
                if (idx < m && g < cap) { st_stream_u64(kout + g, Wk[BP_SWK(idx)]); st_stream_d2(aout + g, La[BP_SWA(idx)]); }
            }
        }
        if (!park) __syncthreads();   // A* | B* and this landing buffer are reused (a parked tile's are not, until it is stored)
    }
    if (PARK && pk_valid) {   // the block's last tile
        __syncthreads();
        if (tid < 32) {
            const u64 ex = lookback_exclusive_2level<false>(status, gstat, pk_tile, ntiles, (u64)pk_total);
            if (tid == 0) {
                s_base = ex;
                if (pk_tile == ntiles - 1) *d_count = ex + (u64)pk_total;
            }
        }
        __syncthreads();
        const u64 base = s_base;
        for (int idx = tid; idx < pk_total; idx += SV_THREADS) {
            const u64 g = base + (u64)idx;
            if (g < cap) { st_stream_u64(kout + g, pk_keys[BP_SWK(idx)]); st_stream_d2(aout + g, pk_amps[BP_SWA(idx)]); }
        }
    }
    if (PRE) {   // block totals, summed in a fixed order (lanes by a fixed tree, warps ascending)
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

template <int MODE, bool FIXED, bool PRE>
static u32 launch_bitpass(const u64* kin, const double2* ain, u64* kout, double2* aout, int p, const GateTab* tab,
                          const PendPred& pend, TileDesc* desc, u64* status, u64* d_count, u64 cap, u32 ntiles, cudaStream_t st,
                          const PreCut* pre = nullptr, double* pre_mass = nullptr, u64* pre_cnt = nullptr) {
    const size_t stg = (size_t)BP_TILE + ((!FIXED && MODE == 1 && PRE && BP_GENP_CTAS < 4) ? BP_PARK_EXTRA : 0);
    const size_t smem = stg * (16 + 16) + (size_t)BP_TILE * 8 + 64 + stg * (8 + 2) +
                        ((!FIXED && MODE == 1 && (PRE ? BP_GENP_CTAS < 4 : BP_GEN2_CTAS < 4)) ? stg * 8 : 0);   // amplitudes x 2, landing keys, A* | B* keys, slots; general one-bit gate: second key array
    static int per_sm[SV_MAX_DEV];
    const u32 grid = sv_launch_persistent(bitpass_kernel<MODE, FIXED, PRE>, per_sm, smem, ntiles, st, kin, ain, kout, aout, p, tab, pend,
                                          (const TileDesc*)desc, status, d_count, cap, ntiles, pre, pre_mass, pre_cnt);
    return grid;
}

int svk_bitpass(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int pair, int fixed,
                const GateTab* tab, const PendPred& pend, TileDesc* desc, u64* status, u32* tile_counter,
                u64* d_count, u64 cap, cudaStream_t st, cudaEvent_t e0, cudaEvent_t e1, const PreCut* pre, double* pre_mass,
                u64* pre_cnt, u32* pre_parts, u32 tnom) {
    (void)tile_counter;
    if (tnom == 0 || tnom > BP_TNOM) tnom = BP_TNOM;
    if (tnom < 256) tnom = 256;
    if (pre_parts) *pre_parts = 0;
    if (n == 0) { cudaMemsetAsync(d_count, 0, sizeof(u64), st); return 0; }
    const u32 ntiles = (u32)((n + tnom - 1) / tnom);
    if (!(pair == 2 || (!pair && fixed)))   // the position-preserving variants have no scan
        cudaMemsetAsync(status, 0, ((size_t)ntiles + (ntiles + 31) / 32 + 8) * sizeof(u64), st);   // tile + group statuses
    int launches = svk_find_splits(kin, n, p, 0, tnom, ntiles, desc, st);
    if (e0) cudaEventRecord(e0, st);
#define SV_BP(P_, F_) launch_bitpass<P_, F_, false>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st)
    if (pair == 2) SV_BP(2, true);                       // monomial blocks: always position preserving
    else if (pair && pre) {
        const u32 g = launch_bitpass<1, false, true>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st, pre, pre_mass, pre_cnt);
        if (pre_parts) *pre_parts = g;
    }
    else if (pair) SV_BP(1, false);
    else { if (fixed) SV_BP(0, true); else SV_BP(0, false); }
#undef SV_BP
    if (e1) cudaEventRecord(e1, st);
    return launches + 1;
}

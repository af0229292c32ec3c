// Diagonal gates and the tile boundaries of the merge passes (row a-4).
// PAPER.md:108-120.
//
// Storage invariant: keys are stored in a permuted ("physical") bit order and kept strictly
// ascending.  A gate never sorts: the qubits on which U actually mixes amplitudes ("active" bits)
// are moved to the least-significant physical positions one at a time, each move being ONE
// streaming pass -- a segmented two-way merge of the bit=0 run and the bit=1 run of every block of
// keys that agree above the moved bit (sv_pair.cu, sv_group.cu).  find_splits cuts such a pass into
// tiles: merge-path splits, one thread per boundary.  Diagonal gates touch amplitudes only.
#include "sv_tile.cuh"

// ---------------------------------------------------------------------------------------
// a-2 diagonal fast path: a <- U[c,c] * a, c = the key's pattern on the gate's qubits
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SV_THREADS) diag_kernel(const u64* __restrict__ keys, double2* __restrict__ amps,
                                                          u64 n, const GateTab* __restrict__ tab) {
    __shared__ double2 d[16];
    __shared__ int cpos[SV_MAX_M];
    __shared__ int mc_s;
    if (threadIdx.x < 16) d[threadIdx.x] = tab->U[threadIdx.x];
    if (threadIdx.x < SV_MAX_M) cpos[threadIdx.x] = tab->ctrl_pos[threadIdx.x];
    if (threadIdx.x == 0) mc_s = tab->mc;
    __syncthreads();
    const int mc = mc_s;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const u64 k = ld_stream_u64(keys + i);
        double2 a = amps[i];
        int cx = 0;
        for (int j = 0; j < mc; ++j) cx |= (int)((k >> cpos[j]) & 1ull) << j;
        const double2 u = d[cx];
        double2 o;
        o.x = __dsub_rn(__dmul_rn(u.x, a.x), __dmul_rn(u.y, a.y));
        o.y = __dadd_rn(__dmul_rn(u.x, a.y), __dmul_rn(u.y, a.x));
        amps[i] = o;
    }
}

int svk_diag(const u64* keys, double2* amps, u64 n, const GateTab* tab, cudaStream_t st) {
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > (u64)sv_sm_count() * 16) blocks = (u64)sv_sm_count() * 16;
    diag_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, tab);
    return 1;
}

// ---------------------------------------------------------------------------------------
// a-3 / f-4: monomial one-bit gate (CNOT, Toffoli, C3X, controlled-Y ...) whose active bit ALREADY sits at the physical
// LSB: partners are stored neighbours, so nothing moves.  PAPER.md:54-55: such a gate "just permutes the amplitudes".
// In place: a tuple with both members and a swapping control pattern trades its two amplitudes (handled by the member
// with bit 0 clear); a lone member of a swapping tuple gets its key's LSB flipped (the order of the array is unchanged:
// its neighbours differ from it above bit 0); phases and a pending truncation (dropped -> dead entry, survivors scaled)
// are applied on the way.  8 B per term when nothing is pending and the entries are unit, else 40 B per term -- against
// 48 B per term for the position-preserving pass that has to move the bit first.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SV_THREADS) perm_lsb_kernel(u64* __restrict__ keys, double2* __restrict__ amps, u64 n,
                                                              const GateTab* __restrict__ gtab, PendPred pd) {
    __shared__ double2 sU[64];
    __shared__ int s_cpos[SV_MAX_M], s_mc, s_sw[16], s_unit;
    if (threadIdx.x < 64) sU[threadIdx.x] = gtab->U[threadIdx.x];
    if (threadIdx.x < SV_MAX_M) s_cpos[threadIdx.x] = gtab->ctrl_pos[threadIdx.x];
    if (threadIdx.x == 0) {
        s_mc = gtab->mc;
        int unit = 1;
        for (int cx = 0; cx < 16; ++cx) {
            const double2* u = &gtab->U[(cx & 15) << 2];
            const int sw = (u[0].x == 0.0 && u[0].y == 0.0) ? 1 : 0;
            s_sw[cx] = sw;
            const double2 x = sw ? u[1] : u[0], y = sw ? u[2] : u[3];
            if (cx < (1 << gtab->mc) && !(x.x == 1.0 && x.y == 0.0 && y.x == 1.0 && y.y == 0.0)) unit = 0;
        }
        s_unit = unit;
    }
    __syncthreads();
    const int mc = s_mc;
    const bool touch_all = pd.active || !s_unit;     // every amplitude changes (scale / phase)
    auto pended = [&](double2 a, u64 key) {
        if (pd.active) {
            if (pend_keep(pd, key, a)) { a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale); }
            else { a.x = 0.0; a.y = 0.0; }
        }
        return a;
    };
    auto times = [&](double2 u, double2 a) {
        if (s_unit) return a;
        const double pr = __dsub_rn(__dmul_rn(u.x, a.x), __dmul_rn(u.y, a.y));
        const double pi = __dadd_rn(__dmul_rn(u.x, a.y), __dmul_rn(u.y, a.x));
        return make_double2(__dadd_rn(0.0, pr), __dadd_rn(0.0, pi));
    };
    // four elements per thread and iteration, all loads of a batch issued before anything is decided
    const u64 chunk = (u64)SV_THREADS * 4;
    const u64 nchunks = (n + chunk - 1) / chunk;
    for (u64 c = blockIdx.x; c < nchunks; c += gridDim.x) {
        u64 k[4], kn[4], kp[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            k[r] = kn[r] = kp[r] = 0;
            if (i < n) { k[r] = keys[i]; kn[r] = (i + 1 < n) ? keys[i + 1] : ~k[r]; kp[r] = (i > 0) ? keys[i - 1] : ~k[r]; }
        }
        int code[4];            // bit 0: swap, bit 1: paired, bit 2: valid; bits 4..: control block
        double2 a[4], an[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            int cx = 0;
            for (int q = 0; q < mc; ++q) cx |= (int)((k[r] >> s_cpos[q]) & 1ull) << q;
            const int b = (int)(k[r] & 1ull);
            const bool paired = b ? (kp[r] == (k[r] & ~1ull)) : (kn[r] == (k[r] | 1ull));
            const int sw = s_sw[cx];
            code[r] = (i < n ? 4 : 0) | (paired ? 2 : 0) | sw | (cx << 4);
            a[r] = an[r] = make_double2(0.0, 0.0);
            if (i < n) {
                const bool owner = sw && paired && !b;                       // trades the tuple's two amplitudes
                const bool self = (sw && !paired) ? touch_all : (!sw && touch_all);
                if (owner || self) a[r] = amps[i];
                if (owner) an[r] = amps[i + 1];
            }
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            if (!(code[r] & 4)) continue;
            const u64 i = c * chunk + (u64)r * SV_THREADS + threadIdx.x;
            const int sw = code[r] & 1, b = (int)(k[r] & 1ull);
            const bool paired = (code[r] & 2) != 0;
            const double2* u = &sU[(code[r] >> 4) << 2];                    // u[row * 2 + col]
            if (sw && paired) {
                if (!b) {
                    const double2 a0 = pended(a[r], k[r]), a1 = pended(an[r], k[r] | 1ull);
                    amps[i] = times(u[1], a1);                               // row 0 <- column 1
                    amps[i + 1] = times(u[2], a0);                           // row 1 <- column 0
                }
            } else if (sw) {                                                 // a lone member moves to the other key of its tuple
                keys[i] = k[r] ^ 1ull;
                if (touch_all) amps[i] = times(u[((b ^ 1) << 1) | b], pended(a[r], k[r]));
            } else if (touch_all) {
                amps[i] = times(u[(b << 1) | b], pended(a[r], k[r]));
            }
        }
    }
}
int svk_perm_lsb(u64* keys, double2* amps, u64 n, const GateTab* tab, const PendPred& pend, cudaStream_t st) {
    if (n == 0) return 0;
    u64 blocks = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (blocks > (u64)sv_sm_count() * 8) blocks = (u64)sv_sm_count() * 8;
    perm_lsb_kernel<<<(unsigned)blocks, SV_THREADS, 0, st>>>(keys, amps, n, tab, pend);
    return 1;
}

// ---------------------------------------------------------------------------------------
// tile boundaries of a bit-move pass (merge-path splits, one thread per boundary)
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ u64 lower_bound_g(const u64* __restrict__ keys, u64 lo, u64 hi, u64 v) {
    while (lo < hi) {
        u64 mid = lo + ((hi - lo) >> 1);
        if (keys[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__global__ void find_splits_kernel(const u64* __restrict__ keys, u64 n, int p, int w, u32 tnom, u32 ntiles,
                                   TileDesc* __restrict__ desc) {
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = j <= ntiles;               // (no early return: the warp shares search results below)
    const bool last = (j >= ntiles);
    const u64 t = last ? n - 1 : (u64)j * tnom;   // n >= 1 here
    const u64 lowmask = (1ull << p) - 1;
    const u64 kt = keys[t];
    const u64 blk = (p == 63) ? 0 : ((kt >> (p + 1)) << (p + 1));
    // block start s, start of its B run mid, block end e: three lower bounds over the globally sorted keys,
    // bracketed by t and advanced TOGETHER so that their dependent loads overlap
    const u64 vmid = blk | (1ull << p);
    const u64 nxt = (p == 63) ? 0 : blk + (2ull << p);
    const bool has_e = (p < 63) && nxt != 0;                    // nxt == 0: wrapped, last block
    // Boundaries of one warp that fall into the same block share s, mid and e: only the first lane of each
    // block searches (its brackets hold for the whole block), the others take its result.
    const int lane = threadIdx.x & 31;
    const unsigned peers = __match_any_sync(0xffffffffu, active ? blk : (~0ull - (u64)lane));
    const int leader = __ffs(peers) - 1;
    const bool searching = active && lane == leader;
    u64 slo = 0, shi = (p == 63) ? 0 : t;                       // keys[t] >= blk: s in [0, t]
    u64 mlo = (kt & (1ull << p)) ? 0 : t + 1, mhi = (kt & (1ull << p)) ? t : n;
    u64 elo = has_e ? t + 1 : n, ehi = n;                       // keys[t] < nxt: e in [t + 1, n]
    if (!searching) { shi = slo; mhi = mlo; ehi = elo; }
    // Bounded gallop from t first: when the blocks are small (the moved bit is low) all three bounds lie within a few
    // elements of t, in cache lines this thread has just touched -- the full-range searches below would instead spend
    // ~28 scattered reads each.  At most 10 doubling steps per bound; the binary searches then start from the brackets.
    {
        const bool mdown = (kt & (1ull << p)) != 0;          // mid lies at or below t
        bool gs = slo < shi, gm = mlo < mhi, ge = elo < ehi;
        for (u64 step = 1; step <= 1024 && (gs || gm || ge); step <<= 1) {
            const u64 cs = (shi > slo + step) ? shi - step : slo;
            const u64 cm = mdown ? ((mhi > mlo + step) ? mhi - step : mlo) : ((mlo + step - 1 < mhi) ? mlo + step - 1 : mhi - 1);
            const u64 ce = (elo + step - 1 < ehi) ? elo + step - 1 : ehi - 1;
            const u64 ks = gs ? keys[cs] : 0, km = gm ? keys[cm] : 0, ke = ge ? keys[ce] : 0;
            if (gs) { if (ks >= blk) { shi = cs; gs = shi > slo; } else { slo = cs + 1; gs = false; } }
            if (gm) {
                if (mdown) { if (km >= vmid) { mhi = cm; gm = mhi > mlo; } else { mlo = cm + 1; gm = false; } }
                else { if (km < vmid) { mlo = cm + 1; gm = mlo < mhi; } else { mhi = cm; gm = false; } }
            }
            if (ge) { if (ke < nxt) { elo = ce + 1; ge = elo < ehi; } else { ehi = ce; ge = false; } }
        }
    }
    while (slo < shi || mlo < mhi || elo < ehi) {
        const u64 sm = slo + ((shi - slo) >> 1), mm = mlo + ((mhi - mlo) >> 1), em = elo + ((ehi - elo) >> 1);
        const u64 ks = (slo < shi) ? keys[sm] : 0, km = (mlo < mhi) ? keys[mm] : 0, ke = (elo < ehi) ? keys[em] : 0;
        if (slo < shi) { if (ks < blk) slo = sm + 1; else shi = sm; }
        if (mlo < mhi) { if (km < vmid) mlo = mm + 1; else mhi = mm; }
        if (elo < ehi) { if (ke < nxt) elo = em + 1; else ehi = em; }
    }
    const u64 s = __shfl_sync(0xffffffffu, slo, leader), mid = __shfl_sync(0xffffffffu, mlo, leader),
              e = __shfl_sync(0xffffffffu, elo, leader);
    if (!active) return;
    TileDesc d;
    d.mid = mid; d.e = e;
    if (last) { d.ia = mid; d.ib = e; desc[j] = d; return; }
    const u64 lenA = mid - s, lenB = e - mid, diag = t - s;
    u64 lo = diag > lenB ? diag - lenB : 0, hi = diag < lenA ? diag : lenA;
    while (lo < hi) {   // A first on ties: A[i] precedes B[diag-1-i] iff lowA <= lowB
        const u64 i = lo + ((hi - lo) >> 1);
        const u64 ka = keys[s + i] & lowmask, kb = keys[mid + (diag - 1 - i)] & lowmask;
        if (ka <= kb) lo = i + 1; else hi = i;
    }
    u64 i = lo, jb = diag - lo;
    if (w >= 0 && (i < lenA || jb < lenB)) {   // do not split a tuple: pull its earlier members across
        u64 nxt;
        if (i < lenA && jb < lenB) {
            const u64 ka = keys[s + i] & lowmask, kb = keys[mid + jb] & lowmask;
            nxt = ka <= kb ? ka : kb;
        } else nxt = (i < lenA) ? (keys[s + i] & lowmask) : (keys[mid + jb] & lowmask);
        const u64 v = nxt >> w;
        while (i > 0 && ((keys[s + i - 1] & lowmask) >> w) == v) --i;
        while (jb > 0 && ((keys[mid + jb - 1] & lowmask) >> w) == v) --jb;
    }
    d.ia = s + i; d.ib = mid + jb;
    desc[j] = d;
}

int svk_find_splits(const u64* keys, u64 n, int p, int w, u32 tnom, u32 ntiles, TileDesc* desc, cudaStream_t st) {
    const u32 nb = (ntiles + 1 + 127) / 128;
    find_splits_kernel<<<nb, 128, 0, st>>>(keys, n, p, w, tnom, ntiles, desc);
    return 1;
}


// ---------------------------------------------------------------------------------------
// tile boundaries of a TWO-bit pass (bits pH > pL moved to the two least-significant positions by ONE streaming pass:
// a four-way merge per tile, sv_dense.cu).  One thread per boundary.
//
// Read a stored key as (high, bH, mid, bL, low) and let rest = (high, mid, low): the pass emits the state in (rest, bH, bL)
// order, so tile j holds the entries whose rank in REST order is in [j tnom, (j + 1) tnom) -- pulled back to the start of a
// tuple.  The boundary is the value R = (h, m, l) of rest with that rank (a selection over the four sorted sub-sequences
// the patterns of (bH, bL) form), found in four steps that only ever take lower bounds over the stored (sorted) keys:
//   (1) the block h of keys that agree above pH, its halves A = [s1, mid1), B = [mid1, e1): the stored position T = j tnom lies
//       in it, and the block holds the same entries in either order, so the rank inside the block is T - s1;
//   (2) m: both halves are sorted by mid -- a merge-path co-rank search on the mid bits gives the mid value of that rank;
//   (3) the sub-blocks (h, 0, m) and (h, 1, m), each a bL = 0 run followed by a bL = 1 run, all four sorted by low;
//   (4) l: the low value of the remaining rank among the four runs, by descent over the bits of low (bits on which all
//       entries still in question agree are skipped; one partition point per run and bit, found together).
// The entries before R are then four stored ranges (TileDesc2); a tile is the difference of two such sets: at most seven
// contiguous pieces.
// ---------------------------------------------------------------------------------------
// K lower bounds over the sorted keys advanced TOGETHER (their dependent loads overlap).  On entry lo[k] <= answer <= hi[k],
// answer = first index in [lo, hi) whose key is >= v[k] (hi if none); hint[k] is a position near it: a bounded gallop from
// the hint brackets the answer before the binary search starts.  On return lo[k] == hi[k] == answer.
template <int K>
__device__ __forceinline__ void multi_lower_bound(const u64* __restrict__ keys, u64 (&lo)[K], u64 (&hi)[K], const u64 (&v)[K],
                                                  const u64 (&hint)[K]) {
    bool go[K], up[K];
    u64 c[K], kk[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        go[k] = lo[k] < hi[k];
        u64 h = hint[k] < lo[k] ? lo[k] : hint[k];
        if (go[k] && h >= hi[k]) h = hi[k] - 1;
        c[k] = h;
    }
#pragma unroll
    for (int k = 0; k < K; ++k) kk[k] = go[k] ? keys[c[k]] : 0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        up[k] = false;
        if (go[k]) {
            if (kk[k] < v[k]) { lo[k] = c[k] + 1; up[k] = true; } else hi[k] = c[k];
            go[k] = lo[k] < hi[k];
        }
    }
    for (u64 step = 1; step <= 2048; step <<= 1) {
        bool any = false;
#pragma unroll
        for (int k = 0; k < K; ++k) any = any || go[k];
        if (!any) break;
#pragma unroll
        for (int k = 0; k < K; ++k)
            c[k] = up[k] ? ((lo[k] + step - 1 < hi[k]) ? lo[k] + step - 1 : hi[k] - 1) : ((hi[k] - lo[k] > step) ? hi[k] - step : lo[k]);
#pragma unroll
        for (int k = 0; k < K; ++k) kk[k] = go[k] ? keys[c[k]] : 0;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (go[k]) {
                if (kk[k] < v[k]) { lo[k] = c[k] + 1; go[k] = up[k] && lo[k] < hi[k]; }
                else { hi[k] = c[k]; go[k] = !up[k] && lo[k] < hi[k]; }
            }
        }
    }
    for (;;) {
        bool any = false;
#pragma unroll
        for (int k = 0; k < K; ++k) any = any || (lo[k] < hi[k]);
        if (!any) break;
#pragma unroll
        for (int k = 0; k < K; ++k) c[k] = lo[k] + ((hi[k] - lo[k]) >> 1);
#pragma unroll
        for (int k = 0; k < K; ++k) kk[k] = (lo[k] < hi[k]) ? keys[c[k]] : 0;
#pragma unroll
        for (int k = 0; k < K; ++k)
            if (lo[k] < hi[k]) { if (kk[k] < v[k]) lo[k] = c[k] + 1; else hi[k] = c[k]; }
    }
}

__global__ void __launch_bounds__(128, 8) find_splits2_kernel(const u64* __restrict__ keys, u64 n, int pH, int pL, int w, u32 tnom, u32 ntiles,
                                    TileDesc2* __restrict__ desc) {
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    TileDesc2 d;
    d.pad_ = 0;
    const u64 T = (u64)j * tnom;
    // (no early return: the boundaries of a warp that fall into the same block / sub-blocks share those searches)
    const bool real = j < ntiles && T < n;
    const int lane = threadIdx.x & 31;
    if (!real && j <= ntiles) { d.p00 = d.m2a = d.p01 = d.m1 = d.p10 = d.m2b = d.p11 = n; desc[j] = d; }
    const u64 bitH = 1ull << pH, bitL = 1ull << pL;             // pL < pH <= 63
    const u64 maskH = (pH == 63) ? 0ull : ~((2ull << pH) - 1);
    const u64 maskL = bitL - 1;
    const u64 maskM = (bitH - 1) & ~((2ull << pL) - 1);
    const u64 kt = real ? keys[T] : 0;
    const u64 hb = kt & maskH;
    // (1) the block of keys that agree above pH.  Only the first lane of every block searches (its brackets, taken from its own
    // T, hold for the block as a whole: s1 <= T', mid1 and e1 anywhere), the others take its result.
    u64 s1, mid1, e1;
    {
        const unsigned peers = __match_any_sync(0xffffffffu, real ? hb : (~0ull - (u64)lane));
        const int leader = __ffs(peers) - 1;
        const bool searching = real && lane == leader;
        const u64 nxt = hb + (bitH << 1);                        // pH == 63: 0
        const bool has_e = (pH < 63) && nxt != 0;                // nxt == 0: wrapped, last block
        const bool inB = (kt & bitH) != 0;
        u64 lo[3] = {0, inB ? 0 : T + 1, has_e ? T + 1 : n};
        u64 hi[3] = {(pH == 63) ? 0 : T, inB ? T : n, n};
        if (!searching) { hi[0] = lo[0]; hi[1] = lo[1]; hi[2] = lo[2]; }
        const u64 v[3] = {hb, hb | bitH, nxt};
        const u64 hint[3] = {T, T, T + 1};
        multi_lower_bound<3>(keys, lo, hi, v, hint);
        s1 = __shfl_sync(0xffffffffu, lo[0], leader); mid1 = __shfl_sync(0xffffffffu, lo[1], leader); e1 = __shfl_sync(0xffffffffu, lo[2], leader);
    }
    if (!real) { s1 = 0; mid1 = 0; e1 = 0; }                     // (idle lanes keep taking part in the shuffles below)
    // (2) co-rank on the mid bits (the bH = 0 half first on ties): the mid value of rank diag inside the block
    const u64 lenA = mid1 - s1, lenB = e1 - mid1, diag = real ? T - s1 : 0;
    u64 ia = 0, jb = 0, m = 0;
    if (real) {
        u64 lo = diag > lenB ? diag - lenB : 0, hi = diag < lenA ? diag : lenA;
        while (lo < hi) {
            const u64 i = lo + ((hi - lo) >> 1);
            const u64 ka = keys[s1 + i] & maskM, kb = keys[mid1 + (diag - 1 - i)] & maskM;
            if (ka <= kb) lo = i + 1; else hi = i;
        }
        ia = lo; jb = diag - lo;
        const bool hasA = ia < lenA, hasB = jb < lenB;           // (one of them: diag < lenA + lenB)
        const u64 ka = hasA ? (keys[s1 + ia] & maskM) : 0, kb = hasB ? (keys[mid1 + jb] & maskM) : 0;
        m = (hasA && (!hasB || ka <= kb)) ? ka : kb;
    }
    // (3) the sub-blocks (h, 0, m) and (h, 1, m): start, start of the bL = 1 run, end
    u64 st[4], en[4];
    {   // (shared by the boundaries of the warp that fall into the same pair of sub-blocks, as in (1))
        const u64 b0 = hb | m, b1 = b0 | bitH;
        const unsigned peers = __match_any_sync(0xffffffffu, real ? b0 : (~0ull - (u64)lane));
        const int leader = __ffs(peers) - 1;
        const bool searching = real && lane == leader;
        u64 lo[6] = {s1, s1, s1, mid1, mid1, mid1};
        u64 hi[6] = {mid1, mid1, mid1, e1, e1, e1};
        const u64 v[6] = {b0, b0 | bitL, b0 + (bitL << 1), b1, b1 | bitL, b1 + (bitL << 1)};
        if (v[5] < b1) lo[5] = hi[5];                            // wrapped: the sub-block ends with the half
        if (!searching) {
#pragma unroll
            for (int k = 0; k < 6; ++k) hi[k] = lo[k];
        }
        const u64 hint[6] = {s1 + ia, s1 + ia, s1 + ia, mid1 + jb, mid1 + jb, mid1 + jb};
        multi_lower_bound<6>(keys, lo, hi, v, hint);
#pragma unroll
        for (int k = 0; k < 6; ++k) lo[k] = __shfl_sync(0xffffffffu, lo[k], leader);
        st[0] = lo[0]; en[0] = lo[1]; st[1] = lo[1]; en[1] = lo[2];
        st[2] = lo[3]; en[2] = lo[4]; st[3] = lo[4]; en[3] = lo[5];
    }
    if (!real) return;
    const u64 diag2 = diag - (st[0] - s1) - (st[2] - mid1);      // rank among the entries of the two sub-blocks, by low
    // (4) the low value of that rank among the four runs
    u64 x[4] = {st[0], st[1], st[2], st[3]};
    u64 l = 0;
    if (pL > 0) {
        u64 lo4[4], hi4[4], fk[4], lk[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) { lo4[c] = st[c]; hi4[c] = en[c]; }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const bool ne = lo4[c] < hi4[c];
            fk[c] = ne ? (keys[lo4[c]] & maskL) : 0; lk[c] = ne ? (keys[hi4[c] - 1] & maskL) : 0;
        }
        u64 prefix = 0;
        int q = pL - 1;
        while (q >= 0) {
            u64 ref = 0, diff = 0;
            bool have = false;
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if (lo4[c] < hi4[c]) {
                    if (!have) { ref = fk[c]; have = true; }
                    diff |= (fk[c] ^ ref) | (lk[c] ^ ref);
                }
            const u64 below_q = (2ull << q) - 1;                 // q <= 61
            diff &= below_q;
            if (diff == 0) { prefix |= ref & below_q; break; }   // every entry still in question has the same low value
            const int nq = 63 - __clzll((long long)diff);
            prefix |= ref & below_q & ~((2ull << nq) - 1);       // the bits they agree on
            q = nq;
            const u64 qb = 1ull << q;
            u64 a[4], b[4];                                      // partition point of every run on bit q: first entry with the bit set
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                a[c] = lo4[c]; b[c] = hi4[c];
                if (a[c] < b[c]) {
                    if (fk[c] & qb) b[c] = a[c];
                    else if (!(lk[c] & qb)) a[c] = b[c];
                    else { a[c] += 1; b[c] -= 1; }
                }
            }
            for (;;) {
                bool any = false;
#pragma unroll
                for (int c = 0; c < 4; ++c) any = any || (a[c] < b[c]);
                if (!any) break;
                u64 mm[4], kk[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) mm[c] = a[c] + ((b[c] - a[c]) >> 1);
#pragma unroll
                for (int c = 0; c < 4; ++c) kk[c] = (a[c] < b[c]) ? keys[mm[c]] : 0;
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    if (a[c] < b[c]) { if (kk[c] & qb) b[c] = mm[c]; else a[c] = mm[c] + 1; }
            }
            u64 below = 0;
#pragma unroll
            for (int c = 0; c < 4; ++c) below += a[c] - st[c];
            const bool one = below <= diag2;                     // the wanted entry has bit q set
            if (one) prefix |= qb;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                if (one) lo4[c] = a[c]; else hi4[c] = a[c];
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const bool ne = lo4[c] < hi4[c];
                if (one) fk[c] = ne ? (keys[lo4[c]] & maskL) : 0; else lk[c] = ne ? (keys[hi4[c] - 1] & maskL) : 0;
            }
            --q;
        }
        l = prefix;
#pragma unroll
        for (int c = 0; c < 4; ++c) x[c] = lo4[c];
        // never split a tuple: its members differ in bH, bL and in the w lowest bits
        const u64 l_al = l & ~((1ull << w) - 1);
        if (l_al != l) {
#pragma unroll
            for (int c = 0; c < 4; ++c)
                while (x[c] > st[c] && (keys[x[c] - 1] & maskL) >= l_al) --x[c];
        }
    }
    d.p00 = x[0]; d.m2a = st[1]; d.p01 = x[1]; d.m1 = mid1; d.p10 = x[2]; d.m2b = st[3]; d.p11 = x[3];
    desc[j] = d;
}

// The tile between boundaries j and j + 1 as contiguous pieces of the input: the difference of two sets of four stored
// ranges each (TileDesc2), at most seven pieces.  One thread per tile; the pass reads the table one tile ahead and only
// has to issue the copies.  Entry (12 words): start index of pieces 0..7, then their lengths (32 bits each; 0 = no piece).
__global__ void make_pieces2_kernel(const TileDesc2* __restrict__ desc, u32 ntiles, u64* __restrict__ table) {
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ntiles) return;
    const TileDesc2 d0 = desc[j], d1 = desc[j + 1];
    const u64 as_[4] = {0, d0.m2a, d0.m1, d0.m2b}, ae_[4] = {d0.p00, d0.p01, d0.p10, d0.p11};
    const u64 bs_[4] = {0, d1.m2a, d1.m1, d1.m2b}, be_[4] = {d1.p00, d1.p01, d1.p10, d1.p11};
    u64 ps[SV_PIECES2];
    u32 pl[SV_PIECES2];
#pragma unroll
    for (int q = 0; q < SV_PIECES2; ++q) { ps[q] = 0; pl[q] = 0; }
    int np = 0;
    u64 last_end = ~0ull;
#pragma unroll
    for (int bi = 0; bi < 4; ++bi) {
        u64 cur = bs_[bi];
        const u64 be = be_[bi];
#pragma unroll
        for (int ai = 0; ai <= 4; ++ai) {
            // the part of [cur, be) before range ai of the earlier boundary (ai == 4: what is left)
            u64 a0 = be, a1 = be;
            if (ai < 4) { a0 = as_[ai]; a1 = ae_[ai]; if (a1 <= a0 || a1 <= cur || a0 >= be) continue; }
            const u64 e = a0 < be ? a0 : be;
            if (e > cur) {
                if (last_end == cur) {            // contiguous with the previous piece
#pragma unroll
                    for (int q = 0; q < SV_PIECES2; ++q) if (q == np - 1) pl[q] += (u32)(e - cur);
                } else {
#pragma unroll
                    for (int q = 0; q < SV_PIECES2; ++q) if (q == np) { ps[q] = cur; pl[q] = (u32)(e - cur); }
                    ++np;
                }
                last_end = e;
            }
            if (ai < 4) { const u64 nx = a1 < be ? a1 : be; if (nx > cur) cur = nx; }
        }
    }
    SV_CHK(np <= SV_PIECES2);
    u64* t = table + (size_t)j * SV_PIECES2_WORDS;
#pragma unroll
    for (int q = 0; q < SV_PIECES2; ++q) t[q] = ps[q];
#pragma unroll
    for (int q = 0; q < SV_PIECES2; q += 2) t[SV_PIECES2 + q / 2] = (u64)pl[q] | ((u64)pl[q + 1] << 32);
}

int svk_find_splits2(const u64* keys, u64 n, int pH, int pL, int w, u32 tnom, u32 ntiles, TileDesc2* desc, cudaStream_t st) {
    const u32 nb = (ntiles + 1 + 127) / 128;
    find_splits2_kernel<<<nb, 128, 0, st>>>(keys, n, pH, pL, w, tnom, ntiles, desc);
    make_pieces2_kernel<<<(ntiles + 127) / 128, 128, 0, st>>>(desc, ntiles, reinterpret_cast<u64*>(desc + ntiles + 1));
    return 2;
}

// Final pass of a gate with MA >= 2 active bits (SURVEY.md rows a-4 .. a-7).
//
// Same tile pipeline as the single-bit pass (sv_pair.cu): persistent blocks, the next tile landing
// through cp.async while the current one is processed, A* | B* partition, one merge-path split per
// thread.  Phase 1 moves the last missing active bit to the LSB (skipped when the active bits
// already sit at physical positions 0 .. MA-1) and leaves the tile in shared memory in its NEW
// order, where the <= 2^MA terms of a tuple are neighbours.  Phase 2:
//   * every term that opens a tuple collects the tuple's presence mask and, from the zero pattern
//     of U, the set of output rows that can be nonzero: the tile's output count is known before
//     any arithmetic, so one scan + look-back fixes every output position;
//   * the outputs are then computed ONE PER THREAD (thread t takes outputs t, t + 256, ... of a round
//     of 2048; the opening terms post (term, row) per output first; column contributions are added in
//     ascending logical column index, every operation rounded separately: DESIGN.md D1) and stored
//     directly, consecutive threads writing consecutive entries.  A row that cancels to exactly 0+0i is written as a dead entry
//     (counted, so the term count stays exact) instead of forcing a second scan.
#include "sv_tile.cuh"
#include "sv_launch.cuh"

//
// PRE (fused apply + truncate, sv_presample.cu): outputs whose probability pattern is below pre->P_floor are not
// written.  Which outputs survive is only known once they are computed: the term that opens a tuple computes the
// tuple's possible rows itself in phase 2a and keeps the SURVIVING rows as the tuple's row mask; the scan, the
// look-back and phase 2b then run on survivors only (a quarter or an eighth of the possible outputs at the cap),
// which phase 2b computes once more, one per thread, and stores densely.
#define GP_ROUND 2048
template <int MA, bool PRE>
__global__ void __launch_bounds__(SV_THREADS, 3) grouppass_kernel(const u64* __restrict__ kin, const double2* __restrict__ ain,
                                                                  u64* __restrict__ kout, double2* __restrict__ aout, int p,
                                                                  const GateTab* __restrict__ gtab, PendPred pd,
                                                                  const TileDesc* __restrict__ desc, u64* status,
                                                                  u64* d_count, u64 cap, u32 ntiles, const PreCut* __restrict__ pre,
                                                                  double* __restrict__ pre_mass, u64* __restrict__ pre_cnt) {
    constexpr int NP = 1 << MA;
    constexpr u64 AM = (u64)NP - 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* La = reinterpret_cast<double2*>(smem_raw);        // landing buffer (next tile)
    double2* sa = La + BP_TILE;                                // work buffer: partitioned tile, then the tile in its new order
    u64* Lk = reinterpret_cast<u64*>(sa + BP_TILE);
    u64* sk = Lk + BP_TILE + 8;
    u64* s_info = sk + BP_TILE;                                // per term: the tuple it opens (rows, masks, control block)
    unsigned short* s_owner = reinterpret_cast<unsigned short*>(s_info + BP_TILE);   // per output of a round: (term << 4) | row
    __shared__ int red[BP_WARPS + 2];
    __shared__ int wc[BP_VT][BP_WARPS];
    __shared__ int s_nA;
    __shared__ u64 s_desc[2][8];
    __shared__ u64 s_base;
    __shared__ __align__(8) u64 s_bar;   // mbarrier of the landing bulk copies
    __shared__ double2 sU[256];
    __shared__ unsigned short s_nzr[16][16];   // [cx][xc]: rows r with U[r][xc] != 0 in control block cx
    __shared__ int s_cpos[SV_MAX_M], s_col[16], s_mc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool mv = p >= 0;
    const u64 Pf = PRE ? pre->P_floor : 0ull;
    double dmass = 0.0;     // PRE: mass and number of the outputs this thread left out (below the floor)
    u32 dcnt = 0;

    for (int i = tid; i < 256; i += SV_THREADS) sU[i] = gtab->U[i];
    if (tid < SV_MAX_M) s_cpos[tid] = gtab->ctrl_pos[tid];
    if (tid < 16) s_col[tid] = gtab->colorder[tid];
    if (tid == 0) s_mc = gtab->mc;
    __syncthreads();
    {
        const int cx = tid >> 4, xc = tid & 15;
        unsigned short m = 0;
        if (cx < (1 << s_mc) && xc < NP)
            for (int r = 0; r < NP; ++r) {
                const double2 u = sU[(((cx << MA) | r) << MA) | xc];
                if (!(u.x == 0.0 && u.y == 0.0)) m |= (unsigned short)(1u << r);
            }
        s_nzr[cx][xc] = m;
    }
    const u64 bit = mv ? (1ull << p) : 0ull;
    const u64 himask = (!mv || p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    u64* gstat = status + ntiles;
    u32 n_dead = 0;

    // The tile lands by bulk copies (TMA): one thread arms the barrier and issues up to six copies (sv_tile.cuh).
    auto issue_loads = [&](const Pieces3& q) {
        if (tid == 0) land_tile_bulk(q, kin, ain, Lk, La, &s_bar);
    };
    if (tid == 0) { mbar_init(&s_bar, 1); fence_proxy_async_smem(); }
    u32 bar_phase = 0;
    const u32 tile0 = first_tile_of_block<!PRE>();
    if (tid < 8) s_desc[0][tid] = reinterpret_cast<const u64*>(desc + tile0)[tid];
    __syncthreads();
    issue_loads(pieces_of(s_desc[0]));
    int par = 0;
    for (u32 tile = tile0; tile < ntiles; tile += gridDim.x, par ^= 1) {
        const u32 next = tile + gridDim.x;
        u64 dnext = 0;
        if (tid < 8 && next < ntiles) dnext = reinterpret_cast<const u64*>(desc + next)[tid];
        const Pieces3 pc = pieces_of(s_desc[par]);
        const int cnt = pc.cnt;
        int nA;
        {   // pick up this thread's landed elements, apply a pending truncation, partition into A* | B*
            mbar_wait(&s_bar, bar_phase);      // the tile has landed
            bar_phase ^= 1u;
            const Landing3 ld = landing_of(pc);
            u64 lk[BP_VT]; double2 la[BP_VT];
#pragma unroll
            for (int r = 0; r < BP_VT; ++r) {
                const int e = tid + r * SV_THREADS;
                lk[r] = 0; la[r] = make_double2(0.0, 0.0);
                if (e < cnt) { lk[r] = Lk[landing_key_slot(pc, ld, e)]; la[r] = La[e]; }
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
            if (!mv || pc.oneblock) {   // load order = A* | B* already (no move: everything is "A", keys unchanged)
                nA = mv ? pc.l0 : cnt;
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    const int e = tid + r * SV_THREADS;
                    if (e < cnt) { sk[e] = lk[r] & ~bit; sa[e] = la[r]; }
                }
            } else {
                u32 balA[BP_VT];
#pragma unroll
                for (int r = 0; r < BP_VT; ++r) {
                    const bool isA = (tid + r * SV_THREADS < cnt) && !(lk[r] & bit);
                    balA[r] = __ballot_sync(0xffffffffu, isA);
                    if (lane == 0) wc[r][warp] = __popc(balA[r]);
                }
                __syncthreads();
                if (warp == 0) {
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
                        sk[slot] = lk[r] & ~bit; sa[slot] = la[r];
                    }
                }
            }
        }
        if (tid < 8 && next < ntiles) s_desc[par ^ 1][tid] = dnext;
        __syncthreads();
        if (next < ntiles) issue_loads(pieces_of(s_desc[par ^ 1]));

        // ---- phase 1: bring the tile into its new order (moved bit at the LSB) ----
        if (mv) {
            const int nB = cnt - nA;
            const u64* skB = sk + nA;
            const double2* saB = sa + nA;
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
            u64 ka = (i < nA) ? sk[i] : ~0ull, kb = (j < nB) ? skB[j] : ~0ull;
            u64 mk[BP_VT]; double2 ma_[BP_VT];
#pragma unroll
            for (int v = 0; v < BP_VT; ++v) {
                mk[v] = 0; ma_[v] = make_double2(0.0, 0.0);
                if (diag + v < endpos) {
                    const bool takeA = ka <= kb;
                    const u64 k = takeA ? ka : kb;
                    ma_[v] = takeA ? sa[i] : saB[j];
                    mk[v] = (k & himask) | ((k & lowmask) << 1) | (takeA ? 0ull : 1ull);
                    if (takeA) { ++i; ka = (i < nA) ? sk[i] : ~0ull; } else { ++j; kb = (j < nB) ? skB[j] : ~0ull; }
                }
            }
            __syncthreads();   // every read of the partitioned tile is done
#pragma unroll
            for (int v = 0; v < BP_VT; ++v)
                if (diag + v < endpos) { sk[diag + v] = mk[v]; sa[diag + v] = ma_[v]; }
            __syncthreads();
        }

        // output row r of the tuple that term e opens (pm: live members, pk: stored members, cx: control block):
        // columns added in ascending LOGICAL index (D1)
        auto tuple_row_x = [&](int e, int r, u32 pm, u32 pk, int cx, double& sr, double& si) {
            const double2* urow = &sU[((cx << MA) | r) << MA];
            sr = 0.0; si = 0.0;
            if ((pm & (pm - 1)) == 0) {                    // a single live member: one product
                const int x = __ffs(pm) - 1;
                const double2 a = sa[e + __popc(pk & ((1u << x) - 1u))];
                const double2 u = urow[x];
                cmul_acc(sr, si, u.x, u.y, a.x, a.y);
            } else {
#pragma unroll
                for (int t = 0; t < NP; ++t) {
                    const int x = s_col[t];
                    if ((pm >> x) & 1u) {
                        const double2 a = sa[e + __popc(pk & ((1u << x) - 1u))];
                        const double2 u = urow[x];
                        cmul_acc(sr, si, u.x, u.y, a.x, a.y);
                    }
                }
            }
        };
        auto tuple_row = [&](int e, int r, double& sr, double& si) {
            const u64 info = s_info[e];
            tuple_row_x(e, r, (u32)((info >> 16) & 0xffffu), (u32)((info >> 32) & 0xffffu), (int)(info >> 48), sr, si);
        };
        // ---- phase 2a: tuples, presence masks, possible output rows -> output counts ----
        const int e0 = min(tid * BP_VT, cnt);
        const int mc = s_mc;
        u64 t_info[BP_VT];   // rows | pm << 16 | pk << 32 | cx << 48 of the tuple a term opens (0: it opens none)
        int mycount = 0;
#pragma unroll
        for (int v = 0; v < BP_VT; ++v) {
            t_info[v] = 0;
            const int e = e0 + v;
            if (e < cnt) {
                const u64 k = sk[e];
                if (e == 0 || (sk[e - 1] >> MA) != (k >> MA)) {   // this term opens a tuple
                    int cx = 0;
                    for (int q = 0; q < mc; ++q) cx |= (int)((k >> s_cpos[q]) & 1ull) << q;
                    u32 pk = 0, pm = 0, rows = 0;
                    for (int w = 0; w < NP && e + w < cnt; ++w) {
                        const u64 kw = sk[e + w];
                        if ((kw >> MA) != (k >> MA)) break;
                        const int x = (int)(kw & AM);
                        pk |= 1u << x;
                        const double2 a = sa[e + w];
                        if (!(a.x == 0.0 && a.y == 0.0)) { pm |= 1u << x; rows |= s_nzr[cx][x]; }
                    }
                    if constexpr (PRE) {   // the rows that survive the floor of the cut that follows: computed here, once more in 2b
                        u32 cand = rows;
                        rows = 0;
                        const bool single = (pm & (pm - 1)) == 0;          // one live member: its amplitude is read once
                        const int x1 = __ffs(pm) - 1;
                        const double2 a1 = single ? sa[e + __popc(pk & ((1u << x1) - 1u))] : make_double2(0.0, 0.0);
                        while (cand) {
                            const int r = __ffs(cand) - 1;
                            cand &= cand - 1;
                            double sr = 0.0, si = 0.0;
                            if (single) {
                                const double2 u = sU[(((cx << MA) | r) << MA) | x1];
                                cmul_acc(sr, si, u.x, u.y, a1.x, a1.y);
                            } else {
                                tuple_row_x(e, r, pm, pk, cx, sr, si);
                            }
                            if (!(sr == 0.0 && si == 0.0)) {       // (an exact cancellation is simply not written)
                                const double pr = prob_of(make_double2(sr, si));
                                if ((u64)__double_as_longlong(pr) >= Pf) rows |= 1u << r;
                                else { dmass = __dadd_rn(dmass, pr); ++dcnt; }
                            }
                        }
                    }
                    t_info[v] = (u64)rows | ((u64)pm << 16) | ((u64)pk << 32) | ((u64)cx << 48);
                    mycount += __popc(rows);
                }
            }
        }
        int total;
        const int excl = block_excl_scan1(mycount, red, &total);
#pragma unroll
        for (int v = 0; v < BP_VT; ++v)
            if (e0 + v < cnt) s_info[e0 + v] = t_info[v];
        // ---- phase 2b: one thread per OUTPUT: consecutive threads write consecutive entries.  Outputs are
        // taken GP_ROUND at a time: the opening terms first post (term, row) for each of their outputs of
        // the round in s_owner, then every thread computes the outputs t, t + 256, ... of the round.  The
        // first round is posted while warp 0 resolves the look-back (one barrier for both) ----
        auto post_round = [&](int h0) {
            if (excl < h0 + GP_ROUND && excl + mycount > h0) {
                int off = excl - h0;
#pragma unroll
                for (int v = 0; v < BP_VT; ++v) {
                    u32 rows = (u32)(t_info[v] & 0xffffu);
                    while (rows) {
                        const int r = __ffs(rows) - 1;
                        rows &= rows - 1;
                        if ((unsigned)off < (unsigned)GP_ROUND) { SV_CHK(e0 + v < cnt); s_owner[off] = (unsigned short)(((e0 + v) << 4) | r); }
                        ++off;
                    }
                }
            }
        };
        if (tid == 0) lookback_publish(status, gstat, tile, ntiles, (u64)total);
        post_round(0);
        if (tid < 32) {
            const u64 ex = lookback_exclusive_2level<false>(status, gstat, tile, ntiles, (u64)total);
            if (tid == 0) {
                s_base = ex;
                if (tile == ntiles - 1) d_count[0] = ex + (u64)total;
            }
        }
        __syncthreads();
        const u64 base = s_base;
        for (int h0 = 0; h0 < total; h0 += GP_ROUND) {
            if (h0 > 0) { post_round(h0); __syncthreads(); }
            const int m = min(total - h0, GP_ROUND);
            for (int q = tid; q < m; q += SV_THREADS) {
                const u32 code = s_owner[q];
                const int e = (int)(code >> 4), r = (int)(code & 15u);
                SV_CHK(e < cnt && r < NP);
                const u64 k = sk[e];
                double sr, si;
                tuple_row(e, r, sr, si);
                if (sr == 0.0 && si == 0.0) ++n_dead;          // exact cancellation: a dead entry
                const u64 g = base + (u64)(h0 + q);
                if (g < cap) { st_stream_u64(kout + g, (k & ~AM) | (u64)r); st_stream_d2(aout + g, make_double2(sr, si)); }
            }
            if (h0 + GP_ROUND < total) __syncthreads();        // s_owner is rewritten by the next round
        }
        __syncthreads();   // the work buffer and the tuple tables are reused by the next tile
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) n_dead += __shfl_xor_sync(0xffffffffu, n_dead, d);
    if (lane == 0 && n_dead) atomicAdd(&d_count[1], (u64)n_dead);
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

// Tile boundaries when no bit has to move (the active bits already sit at positions 0 .. ma-1): nominal
// starts pulled back to the start of a tuple, encoded as one-block descriptors without a B run.
__global__ void find_starts_kernel(const u64* __restrict__ keys, u64 n, int ma, u32 tnom, u32 ntiles, TileDesc* __restrict__ desc) {
    const u32 j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > ntiles) return;
    u64 t = (u64)j * tnom;
    if (t >= n) t = n;
    else if (t > 0) {
        const u64 v = keys[t] >> ma;
        while (t > 0 && (keys[t - 1] >> ma) == v) --t;
    }
    TileDesc d;
    d.ia = t; d.ib = n; d.mid = n; d.e = n;
    desc[j] = d;
}

template <int MA, bool PRE>
static u32 launch_grouppass(const u64* kin, const double2* ain, u64* kout, double2* aout, int p, const GateTab* tab,
                            const PendPred& pend, TileDesc* desc, u64* status, u64* d_count, u64 cap, u32 ntiles, cudaStream_t st,
                            const PreCut* pre = nullptr, double* pre_mass = nullptr, u64* pre_cnt = nullptr) {
    const size_t smem = (size_t)2 * BP_TILE * 24 + 64 + (size_t)BP_TILE * 8 + (size_t)GP_ROUND * 2;   // landing + work + tuple table + owners
    static int per_sm[SV_MAX_DEV];
    const u32 grid = sv_launch_persistent(grouppass_kernel<MA, PRE>, per_sm, smem, ntiles, st, kin, ain, kout, aout, p, tab, pend,
                                          (const TileDesc*)desc, status, d_count, cap, ntiles, pre, pre_mass, pre_cnt);
    return grid;
}

// Final pass of a gate with ma >= 2 active bits.  p < 0: no bit has to move.  Writes the number of
// stored outputs to d_count[0] and the number of dead ones among them (exact cancellations) to d_count[1].
u32 svk_densepass_launch(int ma, bool use_pre, const u64* kin, const double2* ain, u64* kout, double2* aout, int p, const GateTab* tab,
                         const PendPred& pend, TileDesc* desc, u64* status, u64* d_count, u64 cap, u32 ntiles, cudaStream_t st,
                         const PreCut* pre, double* pre_mass, u64* pre_cnt, int maybe_dead, int p2);   // sv_dense.cu

int svk_grouppass(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int ma,
                  const GateTab* tab, const PendPred& pend, TileDesc* desc, u64* status, u64* d_count,
                  u64 cap, cudaStream_t st, cudaEvent_t e0, cudaEvent_t e1, const PreCut* pre, double* pre_mass, u64* pre_cnt,
                  u32* pre_parts, int dense, int maybe_dead, int p2) {
    cudaMemsetAsync(d_count, 0, 2 * sizeof(u64), st);
    if (pre_parts) *pre_parts = 0;
    if (n == 0) return 0;
    const u32 tnom = (u32)(BP_TILE - (1 << ma));
    const u32 ntiles = (u32)((n + tnom - 1) / tnom);
    cudaMemsetAsync(status, 0, ((size_t)ntiles + (ntiles + 31) / 32 + 8) * sizeof(u64), st);
    int launches = 1;
    const bool two = dense && p >= 0 && p2 >= 0 && p2 < p && ma >= 2 && ma <= 4;   // two bits moved by this pass (sv_dense.cu)
    if (two) launches += svk_find_splits2(kin, n, p, p2, ma - 2, tnom, ntiles, reinterpret_cast<TileDesc2*>(desc), st);
    else if (p >= 0) launches += svk_find_splits(kin, n, p, ma - 1, tnom, ntiles, desc, st);
    else { find_starts_kernel<<<(ntiles + 1 + 127) / 128, 128, 0, st>>>(kin, n, ma, tnom, ntiles, desc); launches += 1; }
    if (e0) cudaEventRecord(e0, st);
    if (dense && ma >= 2 && ma <= 4) {   // every entry of U nonzero, no control-like bit: sv_dense.cu
        // (two bits: the pass reads the piece table that follows the ntiles + 1 boundaries)
        TileDesc* dd = two ? reinterpret_cast<TileDesc*>(reinterpret_cast<TileDesc2*>(desc) + ntiles + 1) : desc;
        const u32 g = svk_densepass_launch(ma, pre != nullptr, kin, ain, kout, aout, p, tab, pend, dd, status, d_count, cap, ntiles, st,
                                           pre, pre_mass, pre_cnt, maybe_dead, two ? p2 : -1);
        if (pre && pre_parts) *pre_parts = g;
    } else if (pre) {
        u32 g = 0;
        switch (ma) {
            case 2: g = launch_grouppass<2, true>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st, pre, pre_mass, pre_cnt); break;
            case 3: g = launch_grouppass<3, true>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st, pre, pre_mass, pre_cnt); break;
            default: g = launch_grouppass<4, true>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st, pre, pre_mass, pre_cnt); break;
        }
        if (pre_parts) *pre_parts = g;
    } else {
        switch (ma) {
            case 2: launch_grouppass<2, false>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st); break;
            case 3: launch_grouppass<3, false>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st); break;
            default: launch_grouppass<4, false>(kin, ain, kout, aout, p, tab, pend, desc, status, d_count, cap, ntiles, st); break;
        }
    }
    if (e1) cudaEventRecord(e1, st);
    return launches;
}

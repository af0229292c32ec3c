// Lean single-bit pass (SURVEY.md rows a-3 .. a-7 for gates with ONE active bit, and the
// pure bit moves of wider gates).  PAPER.md:110-120.
//
// Keys are stored ascending in the physical bit order.  Moving physical bit p to the LSB
// is, inside every block of keys that agree above p, a merge of the run with bit p = 0
// ("A") and the run with bit p = 1 ("B") by the bits below p.  The tile (a merge-path
// slice, see find_splits) is loaded in its OLD order, which is ascending in the full key,
// so for a term x the position q of its would-be partner key (x with bit p flipped) is ONE
// binary / galloping search over the tile.  q gives everything the pass needs:
//   * the partner itself (tuple formation), if sk[q] equals that key;
//   * the term's place in the NEW order: with WA[i] / WB[i] the number of outputs led by
//     A / B terms before position i (one packed block scan), an A term at i writes at
//     WA[i] + WB[q] and a B term at i writes at WB[i] + WA[q].
// No sorted copy, no run table, no per-slot loops: each term does one search, the leader
// of a tuple does the 2x2 mat-vec, exact zeros are dropped
// and the outputs go straight to their final, sorted, unique positions.
// A truncation left pending by sv_truncate is applied while loading (dropped terms load
// as 0+0i, survivors are scaled), which removes the separate compaction pass.
#include "sv_device.cuh"

#define BP_VT 4
#define BP_TILE (SV_THREADS * BP_VT)      // 1024 terms per tile
#define BP_TNOM (BP_TILE - 2)             // nominal tile (boundaries are pulled back to a tuple start)

// first index in [lo, hi) with sk[idx] >= key (hi if none); gallops from lo
__device__ __forceinline__ int gallop_lb(const u64* sk, int lo, int hi, u64 key) {
    int step = 1, l = lo, h = lo;
    while (h < hi && sk[h] < key) { l = h + 1; h += step; step <<= 1; }
    if (h > hi) h = hi;
    while (l < h) { const int m = (l + h) >> 1; if (sk[m] < key) l = m + 1; else h = m; }
    return l;
}
// first index in [lo, hi) with sk[idx] >= key, expected near hi; gallops backwards from hi
__device__ __forceinline__ int gallop_lb_back(const u64* sk, int lo, int hi, u64 key) {
    int step = 1, h = hi, l = hi;
    while (l > lo && sk[l - 1] >= key) { h = l - 1; l -= step; step <<= 1; }
    if (l < lo) l = lo;
    while (l < h) { const int m = (l + h) >> 1; if (sk[m] < key) l = m + 1; else h = m; }
    return l;
}

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
                                                                u32* tile_counter, u64* d_count, u64 cap, u32 ntiles) {
    __shared__ __align__(16) double2 sa[BP_TILE];
    __shared__ __align__(16) u64 sk[BP_TILE];
    __shared__ u32 W[BP_TILE + 1];
    __shared__ int red[SV_THREADS / 32 + 2];
    __shared__ u64 s_base;
    __shared__ double2 sU[64];      // [cx][xr][xc], ma = 1: up to 8 control patterns x 4
    __shared__ int s_cpos[SV_MAX_M], s_mc;
    const int tid = threadIdx.x;

    // Tiles are taken in blockIdx order (as CUB's single-pass scan does): a block only ever
    // waits on lower-numbered blocks, which the hardware scheduler has already started.
    const u32 tile = blockIdx.x;
    if (PAIR) {
        if (tid < 64) sU[tid] = gtab->U[tid];
        if (tid < SV_MAX_M) s_cpos[tid] = gtab->ctrl_pos[tid];
        if (tid == 0) s_mc = gtab->mc;
    }
    const TileDesc d0 = desc[tile], d1 = desc[tile + 1];
    u64 ps0, ps1, ps2; int l0, l1, l2;
    if (d0.e == d1.e) { ps0 = d0.ia; l0 = (int)(d1.ia - d0.ia); ps1 = d0.ib; l1 = (int)(d1.ib - d0.ib); ps2 = 0; l2 = 0; }
    else { ps0 = d0.ia; l0 = (int)(d0.mid - d0.ia); ps1 = d0.ib; l1 = (int)(d1.ia - d0.ib); ps2 = d1.mid; l2 = (int)(d1.ib - d1.mid); }
    const int cnt = min(BP_TILE, l0 + l1 + l2);
    {   // coalesced loads of the (up to three) contiguous pieces, all issued before any is used;
        // a pending truncation is applied here (dropped terms become 0+0i, survivors are scaled)
        u64 lk[BP_VT]; double2 la[BP_VT];
#pragma unroll
        for (int r = 0; r < BP_VT; ++r) {
            const int e = tid + r * SV_THREADS;
            if (e < cnt) {
                const u64 g = e < l0 ? ps0 + e : (e < l0 + l1 ? ps1 + (e - l0) : ps2 + (e - l0 - l1));
                lk[r] = ld_stream_u64(kin + g);
                la[r] = ld_stream_d2(ain + g);
            }
        }
#pragma unroll
        for (int r = 0; r < BP_VT; ++r) {
            const int e = tid + r * SV_THREADS;
            if (e < cnt) {
                double2 a = la[r];
                if (pd.active) {
                    if (pend_keep(pd, lk[r], a)) { a.x = __dmul_rn(a.x, pd.scale); a.y = __dmul_rn(a.y, pd.scale); }
                    else { a.x = 0.0; a.y = 0.0; }
                }
                sk[e] = lk[r];
                sa[e] = a;
            }
        }
    }
    __syncthreads();

    const u64 bit = 1ull << p;
    const u64 himask = (p == 63) ? 0 : ~((2ull << p) - 1), lowmask = bit - 1;
    const int i0 = tid * BP_VT;
    u64 ok[BP_VT];            // output base key (new layout, LSB clear) of the element if it leads
    double o0r[BP_VT], o0i[BP_VT], o1r[BP_VT], o1i[BP_VT];
    int qq[BP_VT];            // partner-side position
    u32 wpk[BP_VT];           // packed weight: low 16 = outputs led as an A term, high 16 = as a B term
    u32 sum = 0;
    int qprev = -1; u64 kprev = 0;
#pragma unroll
    for (int v = 0; v < BP_VT; ++v) {
        const int i = i0 + v;
        wpk[v] = 0; qq[v] = 0; ok[v] = 0; o0r[v] = o0i[v] = o1r[v] = o1i[v] = 0.0;
        if (i < cnt) {
            const u64 k = sk[i];
            const double2 a = sa[i];
            const int b = (int)((k >> p) & 1ull);
            const bool same_run = (v > 0) && qprev >= 0 && ((k >> p) == (kprev >> p));
            int q;
            bool has_partner;
            double2 pa = make_double2(0.0, 0.0);
            if (b == 0) {     // partner key k | bit lies after me
                const u64 pk = k | bit;
                q = gallop_lb(sk, same_run ? qprev : i + 1, cnt, pk);
                has_partner = (q < cnt) && (sk[q] == pk);
                if (has_partner) pa = sa[q];
            } else {          // A terms of my block with low <= mine lie before me
                const u64 ak = k & ~bit;
                q = same_run ? gallop_lb(sk, qprev, i, ak + 1) : gallop_lb_back(sk, 0, i, ak + 1);
                has_partner = (q > 0) && (sk[q - 1] == ak);
            }
            qprev = q; kprev = k; qq[v] = q;
            const bool alive = !(a.x == 0.0 && a.y == 0.0);
            const bool palive = has_partner && (b == 1 || !(pa.x == 0.0 && pa.y == 0.0));
            (void)palive;
            u32 w = 0;
            if (PAIR) {
                // the A member leads its tuple; a B term leads only when no A member is stored
                const bool lead = (b == 0) || !has_partner;
                if (lead) {
                    const u64 nk = (k & himask) | ((k & lowmask) << 1);     // new layout, LSB = 0
                    int cx = 0;
                    const int mc = s_mc;
                    for (int j = 0; j < mc; ++j) cx |= (int)((nk >> s_cpos[j]) & 1ull) << j;
                    const double2* u = &sU[cx << 2];                       // u[xr * 2 + xc]
                    double r0 = 0.0, m0 = 0.0, r1 = 0.0, m1 = 0.0;
                    if (b == 0) {
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
                    w = f0 | (f1 << 1);
                    ok[v] = nk; o0r[v] = r0; o0i[v] = m0; o1r[v] = r1; o1i[v] = m1;
                    wpk[v] = (f0 + f1) << (b ? 16 : 0);
                }
            } else {
                if (alive) {
                    ok[v] = (k & himask) | ((k & lowmask) << 1) | (u64)b;
                    o0r[v] = a.x; o0i[v] = a.y;
                    w = 1;
                    wpk[v] = 1u << (b ? 16 : 0);
                }
            }
            qq[v] |= (int)(w << 24) | (b << 23);   // q < 2^11; flags ride in the high bits
            sum += wpk[v];
        }
    }
    int total;
    const u32 excl = (u32)block_excl_scan((int)sum, red, &total);
    {
        u32 run = excl;
#pragma unroll
        for (int v = 0; v < BP_VT; ++v) {
            if (i0 + v < cnt) W[i0 + v] = run;
            run += wpk[v];
        }
        if (tid == 0) W[cnt] = (u32)total;
    }
    const u32 tile_out = ((u32)total & 0xffffu) + ((u32)total >> 16);
    if (tid < 32) {
        const u64 ex = lookback_exclusive_warp(status, tile, (u64)tile_out);
        if (tid == 0) {
            s_base = ex;
            if (tile == ntiles - 1) *d_count = ex + (u64)tile_out;
        }
    }
    __syncthreads();
    const u64 base = s_base;
#pragma unroll
    for (int v = 0; v < BP_VT; ++v) {
        const int i = i0 + v;
        const u32 w = ((u32)qq[v] >> 24) & 3u;
        if (i < cnt && w) {
            const int q = qq[v] & 0x7fffff, b = (qq[v] >> 23) & 1;
            const u32 wi = W[i], wq = W[q];
            const u32 off = b ? ((wi >> 16) + (wq & 0xffffu)) : ((wi & 0xffffu) + (wq >> 16));
            u64 pos = base + off;
            if (PAIR) {
                if (w & 1u) {
                    if (pos < cap) { st_stream_u64(kout + pos, ok[v]); st_stream_d2(aout + pos, make_double2(o0r[v], o0i[v])); }
                    ++pos;
                }
                if (w & 2u) {
                    if (pos < cap) { st_stream_u64(kout + pos, ok[v] | 1ull); st_stream_d2(aout + pos, make_double2(o1r[v], o1i[v])); }
                }
            } else {
                if (pos < cap) { st_stream_u64(kout + pos, ok[v]); st_stream_d2(aout + pos, make_double2(o0r[v], o0i[v])); }
            }
        }
    }
}

int svk_bitpass(const u64* kin, const double2* ain, u64* kout, double2* aout, u64 n, int p, int pair,
                const GateTab* tab, const PendPred& pend, TileDesc* desc, u64* status, u32* tile_counter,
                u64* d_count, u64 cap, cudaStream_t st, cudaEvent_t e0, cudaEvent_t e1) {
    if (n == 0) { cudaMemsetAsync(d_count, 0, sizeof(u64), st); return 0; }
    const u32 ntiles = (u32)((n + BP_TNOM - 1) / BP_TNOM);
    cudaMemsetAsync(status, 0, (size_t)ntiles * sizeof(u64), st);
    cudaMemsetAsync(tile_counter, 0, sizeof(u32), st);
    int launches = svk_find_splits(kin, n, p, 0, BP_TNOM, ntiles, desc, st);
    if (e0) cudaEventRecord(e0, st);
    if (pair) bitpass_kernel<true><<<ntiles, SV_THREADS, 0, st>>>(kin, ain, kout, aout, p, tab, pend, desc, status, tile_counter, d_count, cap, ntiles);
    else bitpass_kernel<false><<<ntiles, SV_THREADS, 0, st>>>(kin, ain, kout, aout, p, tab, pend, desc, status, tile_counter, d_count, cap, ntiles);
    if (e1) cudaEventRecord(e1, st);
    return launches + 1;
}

// Device-side helpers shared by the engine's kernels.
#pragma once
#include "sv_internal.h"

// Checked build (-DSV_CHECKED; python -m paper_2607_07816_b200.build --checked): every index that is computed from data
// is tested against its bound where SV_CHK stands, and the kernel traps on a violation (the launch then fails with an
// error code).  compute-sanitizer is closed on the pool this was developed on; this is what stands in for memcheck.
#ifdef SV_CHECKED
#define SV_CHK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define SV_CHK(cond) do { } while (0)
#endif

#define SV_FLAG_AGG  (1ull << 62)
#define SV_FLAG_INCL (2ull << 62)
#define SV_VAL_MASK  ((1ull << 62) - 1)
#define SV_GRP_ONE   (1ull << 48)            // two-level look-back: one tile's contribution to its group's counter
#define SV_GRP_VAL   ((1ull << 48) - 1)

__device__ __forceinline__ u64 ld_relaxed_u64(const u64* p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u64(u64* p, u64 v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Streaming 128-bit / 64-bit accesses (read once / written once: keep them out of L1).
__device__ __forceinline__ double2 ld_stream_d2(const double2* p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ u64 ld_stream_u64(const u64* p) {
    u64 v;
    asm volatile("ld.global.nc.L1::no_allocate.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream_d2(double2* p, double2 v) {
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
// 256-bit streaming stores (sm_100: STG.256): four keys / two amplitudes, the address 32-byte aligned -- one whole sector
__device__ __forceinline__ void st_stream_u64x4(u64* p, u64 a, u64 b, u64 c, u64 d) {
    asm volatile("st.global.L1::no_allocate.v4.b64 [%0], {%1, %2, %3, %4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory");
}
__device__ __forceinline__ void st_stream_d2x2(double2* p, double ax, double ay, double bx, double by) {
    asm volatile("st.global.L1::no_allocate.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(ax), "d"(ay), "d"(bx), "d"(by) : "memory");
}
__device__ __forceinline__ void st_stream_u64(u64* p, u64 v) {
    asm volatile("st.global.L1::no_allocate.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Decoupled look-back (single-pass chained scan).  Tile ids MUST be handed out by an
// atomic counter so that every predecessor of a running tile has already started.
// Returns the exclusive prefix of `total` over tiles 0..tile-1.  Called by one thread.
__device__ __forceinline__ u64 lookback_exclusive(u64* status, u32 tile, u64 total) {
    if (tile == 0) {
        st_relaxed_u64(&status[0], SV_FLAG_INCL | total);
        return 0;
    }
    st_relaxed_u64(&status[tile], SV_FLAG_AGG | total);
    u64 excl = 0;
    u32 j = tile - 1;
    for (;;) {
        u64 v;
        do { v = ld_relaxed_u64(&status[j]); } while ((v >> 62) == 0);
        excl += v & SV_VAL_MASK;
        if ((v >> 62) == 2) break;
        --j;
    }
    st_relaxed_u64(&status[tile], SV_FLAG_INCL | (excl + total));
    return excl;
}

// Two-level look-back.  A chain of one-warp windows resolves at most 32 tiles per L2 round
// trip; a pass over 2^28 terms has 2.6e5 tiles of ~9000 cycles on ~600 resident blocks, i.e.
// one tile every ~15 cycles -- more than such a chain can carry.  Here tiles are grouped by
// 32.  A tile adds (a) the totals of the tiles before it in its own group and (b) a windowed
// look-back over GROUP statuses, 32 groups (1024 tiles) per round trip; both polls are in
// flight together.  A group's total is gathered by its tiles themselves (one atomic add each: value
// and a count of contributions), so it is complete one round trip after the last of them published
// -- no tile has to close the group; the first tile of the next group later upgrades it to the
// inclusive prefix.  One store and one atomic add to publish, one or two polls to resolve.
//   status[t]   AGG | total of tile t (never overwritten)
//   gstat[g]    sum of the totals published so far (bits 0..47) | how many (bits 48..55; complete at 32),
//               later INCL | inclusive prefix through group g
// Both arrays must be zero at launch.  Called by all 32 lanes of ONE warp.
// PUBLISH = false: the tile's total has been published already (lookback_publish, by one thread, earlier), so that
// other tiles could use it while this block went on with its next tile; this call only resolves the prefix.
__device__ __forceinline__ void lookback_publish(u64* status, u64* gstat, u32 tile, u32 ntiles, u64 total) {
    const u32 g = tile >> 5, r = tile & 31u;
    (void)r; (void)ntiles;
    st_relaxed_u64(&status[tile], SV_FLAG_AGG | total);
    // the group's total is gathered by its 32 tiles themselves: value in bits 0..47, number of tiles that have added
    // theirs in bits 48..55 -- complete, for any reader, one L2 round trip after the last of them published
    atomicAdd(reinterpret_cast<unsigned long long*>(&gstat[g]), (unsigned long long)(total + SV_GRP_ONE));
}
template <bool PUBLISH = true>
__device__ __forceinline__ u64 lookback_exclusive_2level(u64* status, u64* gstat, u32 tile, u32 ntiles, u64 total) {
    const int lane = threadIdx.x & 31;
    const u32 g = tile >> 5, r = tile & 31u;
    if (PUBLISH && lane == 0) lookback_publish(status, gstat, tile, ntiles, total);
    u64 excl = 0;
    bool own_done = (r == 0);
    long long j = (long long)g - 1;          // newest group of the current window
    bool groups_done = (g == 0);
    for (;;) {
        u64 v1 = SV_FLAG_AGG, v2 = SV_FLAG_INCL;
        if (!own_done && lane < (int)r) v1 = ld_relaxed_u64(&status[(g << 5) + lane]);
        const long long idx = j - lane;
        if (!groups_done && idx >= 0) v2 = ld_relaxed_u64(&gstat[idx]);   // virtual groups < 0: inclusive 0
        if (!own_done) {
            if (__all_sync(0xffffffffu, (v1 >> 62) != 0)) {
                u64 c = (lane < (int)r) ? (v1 & SV_VAL_MASK) : 0;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
                excl += c;
                own_done = true;
            }
        }
        if (!groups_done) {
            // a group before this tile's own always has 32 tiles: its total is complete when all 32 have added theirs
            const u32 flagged = __ballot_sync(0xffffffffu, (v2 >> 62) == 2 || ((v2 >> 48) & 0xffull) == 32ull);
            const u32 incl = __ballot_sync(0xffffffffu, (v2 >> 62) == 2);
            const int first = incl ? (__ffs(incl) - 1) : 32;
            const u32 need = (first >= 31) ? 0xffffffffu : ((2u << first) - 1u);
            if ((flagged & need) == need) {
                u64 c = (lane <= first) ? (v2 & SV_GRP_VAL) : 0;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
                excl += c;
                if (first < 32) groups_done = true; else j -= 32;
            }
        }
        if (own_done && groups_done) break;
    }
    if (r == 0 && g > 0 && lane == 0) st_relaxed_u64(&gstat[g - 1], SV_FLAG_INCL | excl);   // = inclusive prefix through group g - 1
    return excl;
}

// Exclusive block scan of one int per thread (blockDim.x == SV_THREADS).  `red` holds
// SV_THREADS/32 + 1 ints.  Returns the exclusive prefix; *total gets the block sum.
__device__ __forceinline__ int block_excl_scan(int v, int* red, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    __syncthreads();  // protect `red` against a previous use
    if (lane == 31) red[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int w = (lane < SV_THREADS / 32) ? red[lane] : 0;
        int winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        if (lane < SV_THREADS / 32) red[lane] = winc - w;
        if (lane == SV_THREADS / 32 - 1) red[SV_THREADS / 32] = winc;
    }
    __syncthreads();
    *total = red[SV_THREADS / 32];
    return red[warp] + inc - v;
}

// The same with ONE barrier: every warp publishes its total, every thread sums the totals of the warps
// before its own.  `red` (SV_THREADS/32 ints) must not be in use by a previous call that other threads
// may still be reading: callers separate two calls by a barrier of their own (the tile loops do).
__device__ __forceinline__ int block_excl_scan1(int v, int* red, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) red[warp] = inc;
    __syncthreads();
    int before = 0, all = 0;
#pragma unroll
    for (int w = 0; w < SV_THREADS / 32; ++w) { const int c = red[w]; all += c; if (w < warp) before += c; }
    *total = all;
    return before + inc - v;
}

// Complex product and accumulation with every operation rounded separately (no FMA):
// the arithmetic contract of DESIGN.md "Determinism" (D1).
__device__ __forceinline__ void cmul_acc(double& sr, double& si, double ur, double ui, double ar, double ai) {
    const double pr = __dsub_rn(__dmul_rn(ur, ar), __dmul_rn(ui, ai));
    const double pi = __dadd_rn(__dmul_rn(ur, ai), __dmul_rn(ui, ar));
    sr = __dadd_rn(sr, pr);
    si = __dadd_rn(si, pi);
}

__device__ __forceinline__ double prob_of(double2 a) {  // p = re*re + im*im, no FMA (D2)
    return __dadd_rn(__dmul_rn(a.x, a.x), __dmul_rn(a.y, a.y));
}

// stored (physical) key -> logical key (see KeyMap): eight cached table reads.
__device__ __forceinline__ u64 logical_key(u64 stored, const KeyMap& km) {
    u64 out = 0;
#pragma unroll
    for (int b = 0; b < 8; ++b) out ^= __ldg(km.lut + b * 256 + (int)((stored >> (8 * b)) & 0xffull));
    return out;
}

// Double-double sums (error-free two_sum): the mass sums of the truncation are taken in this form so that they do not
// depend on the order of summation to within ~2^-100 (D3).
struct dd { double hi, lo; };
__device__ __forceinline__ dd dd_make(double a) { dd r; r.hi = a; r.lo = 0.0; return r; }
__device__ __forceinline__ dd two_sum(double a, double b) {
    dd r; r.hi = __dadd_rn(a, b);
    const double bb = __dsub_rn(r.hi, a);
    r.lo = __dadd_rn(__dsub_rn(a, __dsub_rn(r.hi, bb)), __dsub_rn(b, bb));
    return r;
}
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    s.lo = __dadd_rn(s.lo, __dadd_rn(a.lo, b.lo));
    return two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { b.hi = -b.hi; b.lo = -b.lo; return dd_add(a, b); }
__device__ __forceinline__ bool dd_ge(dd a, dd b) { return a.hi > b.hi || (a.hi == b.hi && a.lo >= b.lo); }

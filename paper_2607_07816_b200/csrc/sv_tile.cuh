// Pieces shared by the tile-pipelined passes (sv_pair.cu, sv_group.cu): tile geometry, the
// asynchronous-copy helpers, tile descriptors -> contiguous pieces, the pending-truncation predicate.
#pragma once
#include "sv_device.cuh"

#ifndef BP_CTAS
#define BP_CTAS 4
#endif
#define BP_VT 4
#define BP_TILE (SV_THREADS * BP_VT)      // 1024 terms per tile
#define BP_TNOM (BP_TILE - 2)             // nominal tile (boundaries are pulled back to a tuple start)
#define BP_WARPS (SV_THREADS / 32)

__device__ __forceinline__ bool pend_keep(const PendPred& pd, u64 stored_key, double2 a) {
    if (a.x == 0.0 && a.y == 0.0) return false;   // dead entry
    const u64 pat = (u64)__double_as_longlong(prob_of(a));
    if (pat > pd.PT) return true;
    if (pat < pd.PT) return false;
    if (pd.KT == ~0ull) return true;
    return logical_key(stored_key, pd.km) <= pd.KT;
}

__device__ __forceinline__ void cp_async8(void* sdst, const void* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(sdst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async16(void* sdst, const void* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(sdst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

struct Pieces3 { u64 ps0, ps1, ps2; int l0, l1, l2, cnt; bool oneblock; };
__device__ __forceinline__ Pieces3 pieces_of(const u64* w) {   // w: desc[tile] (4 words) followed by desc[tile + 1]
    Pieces3 q;
    const u64 ia0 = w[0], ib0 = w[1], mid0 = w[2], e0 = w[3], ia1 = w[4], ib1 = w[5], mid1 = w[6], e1 = w[7];
    q.oneblock = (e0 == e1);
    if (q.oneblock) { q.ps0 = ia0; q.l0 = (int)(ia1 - ia0); q.ps1 = ib0; q.l1 = (int)(ib1 - ib0); q.ps2 = 0; q.l2 = 0; }
    else { q.ps0 = ia0; q.l0 = (int)(mid0 - ia0); q.ps1 = ib0; q.l1 = (int)(ia1 - ib0); q.ps2 = mid1; q.l2 = (int)(ib1 - mid1); }
    q.cnt = min(BP_TILE, q.l0 + q.l1 + q.l2);
    return q;
}


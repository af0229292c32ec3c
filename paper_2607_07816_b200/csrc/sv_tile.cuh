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

// ---- bulk asynchronous copies (TMA, cp.async.bulk) + mbarrier: a tile is at most three CONTIGUOUS pieces of the key and
// of the amplitude array, so one thread lands it with at most six bulk copies instead of one cp.async per element per
// thread: no load instruction, no address arithmetic and no L1TEX traffic on the 256 threads' side.  Source and
// destination must be 16-byte aligned and the size a multiple of 16: amplitudes (16 B) always are; a key piece that
// starts at an odd index is fetched from the even index before it (one key over-fetched in front, possibly one behind),
// see Landing3.
__device__ __forceinline__ void mbar_init(u64* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, u32 parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(a), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* sdst, const void* gsrc, u32 bytes, u64* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"((unsigned)__cvta_generic_to_shared(sdst)), "l"(gsrc), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
// generic-proxy accesses to shared memory made before this point are ordered before later async-proxy (bulk copy) writes
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Tile order of the persistent passes: block b takes tiles first, first + grid, first + 2 grid, ... with first = pi(b), a
// fixed permutation of the blocks (multiplication by a prime modulo the grid size; the identity if the grid size is a
// multiple of it).  Static -- every tile's predecessors belong to blocks that are resident, and the per-block sums of
// the fused call do not depend on timing -- but neighbouring tiles (neighbouring memory, neighbouring look-back words)
// are not worked on by neighbouring SMs at the same moment.  Measured: 2 % faster than first = b for the passes that
// wait in their look-back (general gates, two calls), 1 % slower for those that park their outputs (fused call) and no
// difference for the position-preserving ones: PERMUTE selects it per kernel variant.
#ifndef SV_TILE_MUL
#define SV_TILE_MUL 181u
#endif
template <bool PERMUTE>
__device__ __forceinline__ u32 first_tile_of_block() {
    const u32 G = gridDim.x;
    return (PERMUTE && (G % SV_TILE_MUL)) ? (u32)(((u64)blockIdx.x * SV_TILE_MUL) % G) : blockIdx.x;
}

struct Pieces3 { u64 ps0, ps1, ps2; int l0, l1, l2, cnt; bool oneblock; };
__device__ __forceinline__ Pieces3 pieces_of(const u64* w) {   // w: desc[tile] (4 words) followed by desc[tile + 1]
    Pieces3 q;
    const u64 ia0 = w[0], ib0 = w[1], mid0 = w[2], e0 = w[3], ia1 = w[4], ib1 = w[5], mid1 = w[6], e1 = w[7];
    q.oneblock = (e0 == e1);
    if (q.oneblock) { q.ps0 = ia0; q.l0 = (int)(ia1 - ia0); q.ps1 = ib0; q.l1 = (int)(ib1 - ib0); q.ps2 = 0; q.l2 = 0; }
    else { q.ps0 = ia0; q.l0 = (int)(mid0 - ia0); q.ps1 = ib0; q.l1 = (int)(ia1 - ib0); q.ps2 = mid1; q.l2 = (int)(ib1 - mid1); }
    q.cnt = min(BP_TILE, q.l0 + q.l1 + q.l2);
    SV_CHK(q.l0 >= 0 && q.l1 >= 0 && q.l2 >= 0 && q.l0 + q.l1 + q.l2 <= BP_TILE);
    return q;
}

// Landing slots of a tile that arrived by bulk copies: element e (load order) has its amplitude at La[e] and its key at
// Lk[e + k0] (piece 0), Lk[e + k1] (piece 1) or Lk[e + k2] (piece 2): every key piece starts at an even slot and is
// preceded by the one key that was over-fetched when its first index is odd.  Lk holds BP_TILE + 8 keys.
struct Landing3 { int k0, k1, k2; };
__device__ __forceinline__ Landing3 landing_of(const Pieces3& q) {
    Landing3 L;
    const int o0 = (int)(q.ps0 & 1ull), o1 = (int)(q.ps1 & 1ull), o2 = (int)(q.ps2 & 1ull);
    const int b1 = (q.l0 + o0 + 1) & ~1;                 // slots taken by piece 0 (rounded to an even count)
    const int b2 = b1 + ((q.l1 + o1 + 1) & ~1);
    L.k0 = o0; L.k1 = b1 + o1 - q.l0; L.k2 = b2 + o2 - q.l0 - q.l1;
    return L;
}
__device__ __forceinline__ int landing_key_slot(const Pieces3& q, const Landing3& L, int e) {
    const int sl = e + (e < q.l0 ? L.k0 : (e < q.l0 + q.l1 ? L.k1 : L.k2));
    SV_CHK(sl >= 0 && sl < BP_TILE + 8);
    return sl;
}
// Issued by ONE thread: arm the barrier with the byte count, then the (up to six) copies.
__device__ __forceinline__ void land_tile_bulk(const Pieces3& q, const u64* __restrict__ kin, const double2* __restrict__ ain,
                                               u64* Lk, double2* La, u64* bar) {
    const int o0 = (int)(q.ps0 & 1ull), o1 = (int)(q.ps1 & 1ull), o2 = (int)(q.ps2 & 1ull);
    const int c0 = q.l0 ? ((q.l0 + o0 + 1) & ~1) : 0, c1 = q.l1 ? ((q.l1 + o1 + 1) & ~1) : 0, c2 = q.l2 ? ((q.l2 + o2 + 1) & ~1) : 0;
    const int b1 = (q.l0 + o0 + 1) & ~1, b2 = b1 + ((q.l1 + o1 + 1) & ~1);
    fence_proxy_async_smem();
    mbar_expect_tx(bar, (u32)((c0 + c1 + c2) * 8 + (q.l0 + q.l1 + q.l2) * 16));
    if (q.l0) { bulk_g2s(Lk, kin + (q.ps0 & ~1ull), (u32)c0 * 8u, bar); bulk_g2s(La, ain + q.ps0, (u32)q.l0 * 16u, bar); }
    if (q.l1) { bulk_g2s(Lk + b1, kin + (q.ps1 & ~1ull), (u32)c1 * 8u, bar); bulk_g2s(La + q.l0, ain + q.ps1, (u32)q.l1 * 16u, bar); }
    if (q.l2) { bulk_g2s(Lk + b2, kin + (q.ps2 & ~1ull), (u32)c2 * 8u, bar); bulk_g2s(La + q.l0 + q.l1, ain + q.ps2, (u32)q.l2 * 16u, bar); }
}

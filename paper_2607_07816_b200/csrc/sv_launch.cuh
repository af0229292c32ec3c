// Host-side launch helpers: per-device caches of a kernel's launch attributes, and the cooperative launch of the
// persistent passes.
//
// The tile-pipelined passes (sv_pair.cu, sv_group.cu) are persistent kernels whose blocks wait on one another in the
// decoupled look-back: block b takes tiles b, b + grid, ... and may spin on the status word of a tile another block
// owns.  That is only deadlock free when every block of the grid is resident at the same time.  The grid is sized from
// the occupancy calculator AND launched with cudaLaunchCooperativeKernel: the runtime then either places the whole grid
// at once (waiting for other work on the device to drain if it has to) or fails the launch with an error code --
// a busy device can no longer leave a predecessor block unscheduled while its successors spin.
#pragma once
#include <tuple>
#include <utility>

#include "sv_internal.h"

// Opt-in dynamic shared memory (once per device).  `done` is a per-kernel static bool[SV_MAX_DEV].
template <typename K>
static inline void sv_set_smem_once(K kernel, size_t smem, bool* done) {
    const int dev = sv_cur_device();
    if (!done[dev]) { cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); done[dev] = true; }
}
// Resident blocks per SM of `kernel` (SV_THREADS threads, `smem` dynamic bytes), cached per device in `cache`
// (a per-kernel static int[SV_MAX_DEV]).  Also opts in to the dynamic shared memory size.
template <typename K>
static inline int sv_blocks_per_sm(K kernel, size_t smem, int* cache, int threads = SV_THREADS) {
    const int dev = sv_cur_device();
    if (!cache[dev]) {
        if (smem > 48 * 1024) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        int v = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, kernel, threads, smem) != cudaSuccess || v < 1) v = 1;
        cache[dev] = v;
    }
    return cache[dev];
}
// Cooperative launch of a persistent kernel on min(max_blocks, SMs x resident blocks) blocks.  Returns the grid size
// (0 if the launch failed; the error stays pending for cudaGetLastError).
template <typename... KArgs, typename... Args>
static inline u32 sv_launch_persistent(void (*kernel)(KArgs...), int* per_sm_cache, size_t smem, u32 max_blocks, cudaStream_t st,
                                       Args&&... args) {
    const int per_sm = sv_blocks_per_sm(kernel, smem, per_sm_cache);
    u32 grid = (u32)(sv_sm_count() * per_sm);
    if (grid > max_blocks) grid = max_blocks;
    if (grid == 0) return 0;
    std::tuple<KArgs...> t(std::forward<Args>(args)...);
    cudaError_t e = std::apply([&](auto&... a) {
        void* p[] = {(void*)&a...};
        return cudaLaunchCooperativeKernel((const void*)kernel, dim3(grid), dim3(SV_THREADS), p, smem, st);
    }, t);
    return e == cudaSuccess ? grid : 0;
}

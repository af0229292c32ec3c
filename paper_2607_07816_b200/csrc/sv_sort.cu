// LSD radix sort of (uint64 key, uint32 value) pairs, 8 bits per pass, stable; plus the
// small gather kernels of the load / readout paths (SURVEY.md row a-11 and sv_load).
// Used off the gate hot path: to establish the sorted storage order when a state is
// loaded and to order the k records sv_top returns by (p desc, key asc).
#include "sv_device.cuh"

#define RS_ITEMS 8
#define RS_TILE (SV_THREADS * RS_ITEMS)
#define RS_WARPS (SV_THREADS / 32)

__global__ void __launch_bounds__(SV_THREADS) rs_hist_kernel(const u64* __restrict__ keys, u64 n, int shift, u32 ntiles,
                                                             u32* __restrict__ counts) {
    __shared__ u32 h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const u64 t0 = (u64)blockIdx.x * RS_TILE;
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) {
        const u64 i = t0 + (u64)r * SV_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&h[(u32)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    counts[(u64)threadIdx.x * ntiles + blockIdx.x] = h[threadIdx.x];
}

// in-place exclusive scan of u32 (decoupled look-back), 2048 entries per tile
__global__ void __launch_bounds__(SV_THREADS) rs_scan_kernel(u32* __restrict__ data, u64 n, u64* status, u32* tile_counter) {
    __shared__ int red[SV_THREADS / 32 + 2];
    __shared__ u32 s_tile;
    __shared__ u64 s_base;
    if (threadIdx.x == 0) s_tile = atomicAdd(tile_counter, 1u);
    __syncthreads();
    const u32 tile = s_tile;
    const u64 i0 = (u64)tile * RS_TILE + (u64)threadIdx.x * RS_ITEMS;
    u32 v[RS_ITEMS];
    int sum = 0;
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) { v[r] = (i0 + r < n) ? data[i0 + r] : 0u; sum += (int)v[r]; }
    int total;
    const int excl = block_excl_scan(sum, red, &total);
    if (threadIdx.x == 0) s_base = lookback_exclusive(status, tile, (u64)(u32)total);
    __syncthreads();
    u32 run = (u32)s_base + (u32)excl;
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) {
        if (i0 + r < n) data[i0 + r] = run;
        run += v[r];
    }
}

__global__ void __launch_bounds__(SV_THREADS) rs_scatter_kernel(const u64* __restrict__ kin, const u32* __restrict__ vin,
                                                                u64* __restrict__ kout, u32* __restrict__ vout, u64 n,
                                                                int shift, u32 ntiles, const u32* __restrict__ offsets) {
    __shared__ u32 cntw[RS_WARPS][256];
    __shared__ u32 gbase[256];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int w = 0; w < RS_WARPS; ++w) cntw[w][tid] = 0;
    __syncthreads();
    const u64 wbase = (u64)blockIdx.x * RS_TILE + (u64)warp * (32 * RS_ITEMS);
    u64 k[RS_ITEMS]; u32 lr[RS_ITEMS];
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) {
        const u64 i = wbase + (u64)r * 32 + lane;
        const bool valid = i < n;
        k[r] = valid ? kin[i] : 0;
        const u32 d = valid ? ((u32)(k[r] >> shift) & 255u) : 256u;
        const u32 peers = __match_any_sync(0xffffffffu, d);
        const u32 before = __popc(peers & ((1u << lane) - 1u));
        u32 prev = 0;
        if (valid) prev = cntw[warp][d];
        __syncwarp();
        if (valid && before == 0) cntw[warp][d] = prev + __popc(peers);
        __syncwarp();
        lr[r] = prev + before;
    }
    __syncthreads();
    {   // exclusive scan over warps for digit = tid, and the tile's global base for that digit
        u32 run = 0;
        for (int w = 0; w < RS_WARPS; ++w) { const u32 c = cntw[w][tid]; cntw[w][tid] = run; run += c; }
        gbase[tid] = offsets[(u64)tid * ntiles + blockIdx.x];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RS_ITEMS; ++r) {
        const u64 i = wbase + (u64)r * 32 + lane;
        if (i < n) {
            const u32 d = (u32)(k[r] >> shift) & 255u;
            const u64 pos = (u64)gbase[d] + cntw[warp][d] + lr[r];
            kout[pos] = k[r];
            vout[pos] = vin[i];
        }
    }
}

// In-place exclusive scan of n u32 values.  status: (n / 2048 + 2) u64 words of scratch.
int svk_scan_u32(u32* data, u64 n, u64* status, u32* tile_counter, cudaStream_t st) {
    if (n == 0) return 0;
    const u32 nscan = (u32)((n + RS_TILE - 1) / RS_TILE);
    cudaMemsetAsync(status, 0, (size_t)nscan * 8 + 8, st);
    cudaMemsetAsync(tile_counter, 0, sizeof(u32), st);
    rs_scan_kernel<<<nscan, SV_THREADS, 0, st>>>(data, n, status, tile_counter);
    return 1;
}

size_t svk_sort_scratch_bytes(u64 n) {
    const u64 ntiles = (n + RS_TILE - 1) / RS_TILE + 1;
    const u64 ncounts = 256 * ntiles;
    const u64 nscan = (ncounts + RS_TILE - 1) / RS_TILE + 1;
    return (size_t)(ncounts * 4 + 256 + nscan * 8 + 256);
}

// Sorts n pairs ascending by the low `bits` bits of the key.  Ping-pongs between the two
// buffer pairs; *result_in_alt tells where the result ended.  n < 2^32.
int svk_sort_pairs(u64* keys, u32* vals, u64* keys_alt, u32* vals_alt, u64 n, int bits, u32* scratch, cudaStream_t st,
                   int* result_in_alt) {
    *result_in_alt = 0;
    if (n <= 1 || bits <= 0) return 0;
    const u32 ntiles = (u32)((n + RS_TILE - 1) / RS_TILE);
    const u64 ncounts = 256ull * ntiles;
    const u32 nscan = (u32)((ncounts + RS_TILE - 1) / RS_TILE);
    u32* counts = scratch;
    u64* status = reinterpret_cast<u64*>(reinterpret_cast<unsigned char*>(scratch) + ((ncounts * 4 + 255) / 256) * 256);
    u32* tile_counter = reinterpret_cast<u32*>(status + nscan);
    int launches = 0, flip = 0;
    for (int shift = 0; shift < bits; shift += 8) {
        u64* ki = flip ? keys_alt : keys; u32* vi = flip ? vals_alt : vals;
        u64* ko = flip ? keys : keys_alt; u32* vo = flip ? vals : vals_alt;
        rs_hist_kernel<<<ntiles, SV_THREADS, 0, st>>>(ki, n, shift, ntiles, counts);
        cudaMemsetAsync(status, 0, (size_t)nscan * 8 + 8, st);
        rs_scan_kernel<<<nscan, SV_THREADS, 0, st>>>(counts, ncounts, status, tile_counter);
        rs_scatter_kernel<<<ntiles, SV_THREADS, 0, st>>>(ki, vi, ko, vo, n, shift, ntiles, counts);
        launches += 3;
        flip ^= 1;
    }
    *result_in_alt = flip;
    return launches;
}

__global__ void iota_kernel(u32* v, u64 n) {
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) v[i] = (u32)i;
}
__global__ void gather_u64_kernel(const u64* __restrict__ src, const u32* __restrict__ idx, u64* __restrict__ dst, u64 n, int invert) {
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const u64 v = src[idx[i]];
        dst[i] = invert ? ~v : v;
    }
}
__global__ void gather_c128_kernel(const double2* __restrict__ src, const u32* __restrict__ idx, double2* __restrict__ dst, u64 n) {
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = src[idx[i]];
}
__global__ void pat_to_prob_kernel(const u64* __restrict__ pat, double* __restrict__ prob, u64 n) {
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        prob[i] = __longlong_as_double((long long)pat[i]);
}
static unsigned grid_for(u64 n) {
    u64 b = (n + SV_THREADS * 4 - 1) / (SV_THREADS * 4);
    if (b > (u64)sv_sm_count() * 8) b = (u64)sv_sm_count() * 8;
    if (b < 1) b = 1;
    return (unsigned)b;
}
int svk_iota(u32* v, u64 n, cudaStream_t st) { if (!n) return 0; iota_kernel<<<grid_for(n), SV_THREADS, 0, st>>>(v, n); return 1; }
int svk_gather_u64(const u64* src, const u32* idx, u64* dst, u64 n, int invert, cudaStream_t st) {
    if (!n) return 0; gather_u64_kernel<<<grid_for(n), SV_THREADS, 0, st>>>(src, idx, dst, n, invert); return 1;
}
int svk_gather_c128(const double2* src, const u32* idx, double2* dst, u64 n, cudaStream_t st) {
    if (!n) return 0; gather_c128_kernel<<<grid_for(n), SV_THREADS, 0, st>>>(src, idx, dst, n); return 1;
}
int svk_pat_to_prob(const u64* pat, double* prob, u64 n, cudaStream_t st) {
    if (!n) return 0; pat_to_prob_kernel<<<grid_for(n), SV_THREADS, 0, st>>>(pat, prob, n); return 1;
}

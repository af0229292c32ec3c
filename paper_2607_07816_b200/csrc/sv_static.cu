// sv_norm_static (include/sparse_sv_static.h): the mass of a term array (Eq. 4) for
// callers that may not allocate -- under CUDA graph capture, in serving loops, in harnesses that forbid cudaMalloc.
//
// A variant of the norm of sv_select.cu (norm_partial_kernel / norm_final_kernel / svk_norm) whose partial sums live
// in a file-scope device array instead of the handle's arena.  Grid, strides and the order of every addition are
// those of svk_norm (keep the two in step): same bits as sv_norm on the same amplitude array.
//
// The array is shared by every call on a device and keeps the last call's contents.  Nothing has to start at zero:
// the final kernel reads partials [0, nb) and the partial kernel of the same call, earlier on the same stream, wrote
// exactly those.  Calls that overlap on the GPU race on it (documented in the header).
//
// In host code `g_norm_scratch` is a host-side stand-in for the symbol, NOT a device address: the kernels get the
// address cudaGetSymbolAddress returns, looked up once per device with that device current.
#include <cstdio>
#include <mutex>

#include "../../include/sparse_sv_static.h"
#include "sv_device.cuh"

#define SV_NORM_STATIC_BLOCKS 1024
static_assert(SV_NORM_STATIC_BLOCKS * sizeof(double) == SV_NORM_STATIC_SCRATCH_BYTES, "scratch size stated in the header");

static __device__ __align__(256) double g_norm_scratch[SV_NORM_STATIC_BLOCKS];

static __global__ void __launch_bounds__(SV_THREADS) norm_partial_static_kernel(const double2* __restrict__ amps, u64 n,
                                                                                double* __restrict__ partials) {
    __shared__ double red[SV_THREADS];
    double s = 0.0;
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) s = __dadd_rn(s, prob_of(ld_stream_d2(amps + i)));
    red[threadIdx.x] = s;
    __syncthreads();
    for (int d = SV_THREADS / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) red[threadIdx.x] = __dadd_rn(red[threadIdx.x], red[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = red[0];
}
static __global__ void __launch_bounds__(SV_THREADS) norm_final_static_kernel(const double* __restrict__ partials, int nb,
                                                                              double* __restrict__ out) {
    __shared__ double red[SV_THREADS];
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += SV_THREADS) s = __dadd_rn(s, partials[i]);
    red[threadIdx.x] = s;
    __syncthreads();
    for (int d = SV_THREADS / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) red[threadIdx.x] = __dadd_rn(red[threadIdx.x], red[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = red[0];
}

static thread_local const char* t_err = "";
static thread_local char t_errbuf[192];

static int fail(int code, const char* what, cudaError_t e = cudaSuccess) {
    if (e != cudaSuccess) {
        snprintf(t_errbuf, sizeof(t_errbuf), "%s: %s", what, cudaGetErrorString(e));
        t_err = t_errbuf;
    } else {
        t_err = what;
    }
    return code;
}

// device address of g_norm_scratch, per device
static double* g_scratch_ptr[SV_MAX_DEV];
static std::mutex g_scratch_mu;

static int scratch_of_current_device(double** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(SV_ERR_CUDA, "sv_norm_static: cudaGetDevice", e);
    if (dev < 0 || dev >= SV_MAX_DEV) return fail(SV_ERR_CUDA, "sv_norm_static: device ordinal beyond the per-device table");
    std::lock_guard<std::mutex> lk(g_scratch_mu);
    if (!g_scratch_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_norm_scratch);
        if (e != cudaSuccess || !p) return fail(SV_ERR_CUDA, "sv_norm_static: cudaGetSymbolAddress of the scratch array", e);
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return SV_OK;
}

// nonzero: CUDA knows the pointer as plain (unregistered) host memory
static int plain_host_pointer(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return at.type == cudaMemoryTypeUnregistered;
}

extern "C" int sv_norm_static_init(void) {
    t_err = "";
    double* p = nullptr;
    return scratch_of_current_device(&p);
}

extern "C" const char* sv_static_last_error(void) { return t_err; }

extern "C" int sv_norm_static(const sv_c128* dev_amps, uint64_t n, double* dev_mass, void* stream) {
    t_err = "";
    if (n > SV_NORM_STATIC_MAX_TERMS) return fail(SV_ERR_INVALID_ARG, "sv_norm_static: n exceeds SV_NORM_STATIC_MAX_TERMS (2^32 terms)");
    if (!dev_mass || ((uintptr_t)dev_mass & 7)) return fail(SV_ERR_INVALID_ARG, "sv_norm_static: dev_mass is null or not 8-byte aligned");
    if (n && (!dev_amps || ((uintptr_t)dev_amps & 15))) return fail(SV_ERR_INVALID_ARG, "sv_norm_static: dev_amps is null or not 16-byte aligned");
    if (plain_host_pointer(dev_mass) || (n && plain_host_pointer(dev_amps)))
        return fail(SV_ERR_INVALID_ARG, "sv_norm_static: a pointer is plain host memory (device pointers are required)");
    double* partials = nullptr;
    const int rc = scratch_of_current_device(&partials);
    if (rc != SV_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    int nb = (int)((n + SV_THREADS * 8 - 1) / (SV_THREADS * 8));     // the grid of svk_norm
    if (nb < 1) nb = 1;
    if (nb > SV_NORM_STATIC_BLOCKS) nb = SV_NORM_STATIC_BLOCKS;
    norm_partial_static_kernel<<<nb, SV_THREADS, 0, st>>>(reinterpret_cast<const double2*>(dev_amps), (u64)n, partials);
    norm_final_static_kernel<<<1, SV_THREADS, 0, st>>>(partials, nb, dev_mass);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SV_ERR_CUDA, "sv_norm_static: kernel launch", e);
    return SV_OK;
}

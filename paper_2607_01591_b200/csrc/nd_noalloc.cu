// nd_noalloc.cu -- nd_fission_rate_static: the fission rate F = sum_r A~_r sum_g nuSigma_f[m(r)][g] phi[r][g] (the k_eff update of
// Eq. (1); row A6 of DESIGN.md) for callers that can neither allocate nor hand over a workspace: code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The existing path (nd_source_update's
// d_fission_rate_out) keeps its per-block partial sums in the problem's caller-owned workspace; here they live in a
// file-scope __device__ array of a fixed, stated size, which every GPU that loads the library holds until the process exits.
//
// Two stages, both with a FIXED decomposition, so the result does not depend on the number of SMs or on the grid:
//   stage 1: block b adds the kChunk consecutive elements [b kChunk, (b+1) kChunk) of the flattened [R][G] array
//            (thread t: elements t, t + 256, ..., then a shuffle / shared-memory tree) -> scratch[b]
//   stage 2: one block adds scratch[0 .. n_blocks) (thread t: t, t + 1024, ..., then the same tree) -> *d_fission_rate_out
// Stage 2 reads exactly the entries stage 1 of the same call wrote: nothing has to start at zero and nothing is cleared.  The
// array is SHARED by every call on the device and keeps the last call's partial sums: two calls that overlap on the GPU
// (different streams, or graphs replayed concurrently) race on it.
//
// The name of a __device__ array is, in host code, a host-side stand-in and not a device address; the address the kernels get
// comes from cudaGetSymbolAddress, asked once per device with that device current (below).
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "nd.h"
#include "nd_internal.h"

namespace {

constexpr int kChunk = 4096;                                               // elements of [R][G] per stage-1 block
constexpr long long kScratchDoubles = ND_STATIC_FISSION_MAX_ELEMENTS / kChunk;   // 32768 doubles = 256 KiB per device
constexpr int kMaxDevices = 64;

static __device__ __align__(256) double g_fission_scratch[kScratchDoubles];

__device__ __forceinline__ double block_sum_fixed(double v, double* sh)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = v;
    __syncthreads();
    if (w == 0) {
        v = lane < (int)(blockDim.x >> 5) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;   // valid in thread 0
}

__global__ void __launch_bounds__(256) k_fission_chunks(const double* __restrict__ phi, const int32_t* __restrict__ reg_mat,
                                                        const double* __restrict__ nusf, const double* __restrict__ vol,
                                                        double* __restrict__ scratch, long long n, int G)
{
    __shared__ double sh[32];
    const long long i0 = (long long)blockIdx.x * kChunk;
    double s = 0.0;
#pragma unroll 4
    for (int j = threadIdx.x; j < kChunk; j += 256) {
        const long long i = i0 + j;
        if (i < n) {
            const long long r = i / G;
            const int g = (int)(i - r * G);
            s += vol[r] * nusf[(size_t)reg_mat[r] * G + g] * phi[i];
        }
    }
    s = block_sum_fixed(s, sh);
    if (threadIdx.x == 0) scratch[blockIdx.x] = s;
}

__global__ void __launch_bounds__(1024) k_fission_total(const double* __restrict__ scratch, int n_blocks, double* __restrict__ out)
{
    __shared__ double sh[32];
    double s = 0.0;
    for (int b = threadIdx.x; b < n_blocks; b += 1024) s += scratch[b];
    s = block_sum_fixed(s, sh);
    if (threadIdx.x == 0) *out = s;
}

// device address of g_fission_scratch on every device that has asked for it
std::mutex g_mu;
double* g_scratch_ptr[kMaxDevices] = {};

nd_status scratch_of_current_device(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return nd_fail(ND_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return nd_fail(ND_ERR_RANGE, "nd_fission_rate_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_fission_scratch);   // of the CURRENT device
        if (e != cudaSuccess || !p) {
            char buf[256];
            snprintf(buf, sizeof buf, "cudaGetSymbolAddress(g_fission_scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
            return nd_fail(ND_ERR_CUDA, buf);
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return ND_OK;
}

} // namespace

extern "C" nd_status nd_fission_rate_static(int32_t n_regions, int32_t n_groups, const double* d_phi, const int32_t* d_region_material,
                                            const double* d_nu_sigma_f, const double* d_volume, double* d_fission_rate_out,
                                            void* cuda_stream)
{
    if (!d_phi || !d_region_material || !d_nu_sigma_f || !d_volume || !d_fission_rate_out)
        return nd_fail(ND_ERR_NULL, "nd_fission_rate_static: NULL argument");
    if (n_regions < 1 || n_groups < 1) return nd_fail(ND_ERR_INVALID, "nd_fission_rate_static: n_regions and n_groups must be >= 1");
    const long long n = (long long)n_regions * n_groups;
    if (n > ND_STATIC_FISSION_MAX_ELEMENTS) {
        char buf[256];
        snprintf(buf, sizeof buf, "nd_fission_rate_static: n_regions * n_groups = %lld exceeds ND_STATIC_FISSION_MAX_ELEMENTS = %lld "
                 "(the static scratch holds one partial sum per %d elements); use nd_source_update with a workspace",
                 n, (long long)ND_STATIC_FISSION_MAX_ELEMENTS, kChunk);
        return nd_fail(ND_ERR_RANGE, buf);
    }
    double* scratch = nullptr;
    const nd_status rc = scratch_of_current_device(&scratch);
    if (rc != ND_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const int n_blocks = (int)((n + kChunk - 1) / kChunk);
    k_fission_chunks<<<n_blocks, 256, 0, st>>>(d_phi, d_region_material, d_nu_sigma_f, d_volume, scratch, n, n_groups);
    k_fission_total<<<1, 1024, 0, st>>>(scratch, n_blocks, d_fission_rate_out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return nd_fail(ND_ERR_CUDA, cudaGetErrorString(e));
    return ND_OK;
}

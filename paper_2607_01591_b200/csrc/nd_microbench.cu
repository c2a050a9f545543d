// nd_microbench.cu -- the two micro-benchmarks behind the roofline denominators of DESIGN.md section 5 (SURVEY 8(d):
// "measure both ... before quoting any roofline fraction"):
//   * MUFU.EX2 issue rate per clock per SM -- one Eq.-(5) update needs exactly one, so
//     n_SM x rate x clock is the ceiling of the sweep in updates per second;
//   * FP64 RED (atomic add without return) throughput on random 256-byte rows, L2-resident and HBM-resident -- what the
//     tally flush of the sweep can expect from the memory system.
// Diagnostics only: nothing of the hot path calls this.
#include <cstdio>

#include <cuda_runtime.h>

#include "nd.h"
#include "nd_internal.h"

namespace {

constexpr int kChains = 8;   // independent ex2 chains per thread: more than the MUFU latency / issue interval needs

// Every thread runs kChains independent chains x <- 2^x - 1 (stays in [-0.5, 0]); the FADD runs on the FMA pipe (128 lanes per
// clock per SM), so the XU pipe (MUFU) is the only one that saturates.  One block of 1024 threads per SM.
__global__ void __launch_bounds__(1024) k_mufu_rate(int iters, float seed, float* __restrict__ sink, long long* __restrict__ cycles,
                                                   unsigned long long* __restrict__ nanos, unsigned* __restrict__ smid)
{
    float x[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = seed - 0.01f * (float)c - 1e-4f * (float)(threadIdx.x & 31);
    __syncthreads();
    unsigned long long n0, n1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(n0));
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < kChains; ++c) {
            float y;
            asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x[c]));
            x[c] = y - 1.0f;
        }
    }
    __syncthreads();
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(n1));
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c];
    if (s == 12345.678f) sink[0] = s;   // keeps the chains alive
    if (threadIdx.x == 0) {
        cycles[blockIdx.x] = t1 - t0;
        nanos[blockIdx.x] = n1 - n0;
        unsigned id;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(id));
        smid[blockIdx.x] = id;
    }
}

// One warp instruction = 32 lanes adding to the 32 doubles of one pseudo-randomly chosen 256-byte row of `table`.
__global__ void __launch_bounds__(256) k_red_rate(double* __restrict__ table, unsigned n_rows_mask, int iters)
{
    const unsigned lane = threadIdx.x & 31u;
    unsigned h = (blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        h = h * 1664525u + 1013904223u;
        const unsigned row = (h >> 7) & n_rows_mask;
        atomicAdd(table + (size_t)row * 32u + lane, 1.0);
    }
}

#define MB_CUDA(call)                                                                                    \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            char buf_[384];                                                                              \
            snprintf(buf_, sizeof buf_, "nd_microbench: %s failed: %s", #call, cudaGetErrorString(e_)); \
            if (ev0) cudaEventDestroy(ev0);                                                              \
            if (ev1) cudaEventDestroy(ev1);                                                              \
            return nd_fail(ND_ERR_CUDA, buf_);                                                           \
        }                                                                                                \
    } while (0)

} // namespace

extern "C" nd_status nd_microbench(void* device_workspace, size_t device_bytes, void* cuda_stream, nd_microbench_result* out)
{
    if (!device_workspace || !out) return nd_fail(ND_ERR_NULL, "nd_microbench: NULL argument");
    if (reinterpret_cast<uintptr_t>(device_workspace) % 256 != 0) return nd_fail(ND_ERR_WORKSPACE, "nd_microbench: workspace must be 256-byte aligned");
    if (device_bytes < ((size_t)64 << 20)) return nd_fail(ND_ERR_WORKSPACE, "nd_microbench: workspace must hold at least 64 MiB");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    int dev = 0, n_sm = 0, major = 0;
    MB_CUDA(cudaGetDevice(&dev));
    MB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    MB_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return nd_fail(ND_ERR_CUDA, "nd_microbench: libnd_moc.so holds sm_100a kernels only");
    if (n_sm > 1024) n_sm = 1024;
    MB_CUDA(cudaEventCreate(&ev0));
    MB_CUDA(cudaEventCreate(&ev1));
    nd_microbench_result r{};
    r.n_sm = n_sm;

    // ---- MUFU.EX2 ----
    char* ws = static_cast<char*>(device_workspace);
    float* sink = reinterpret_cast<float*>(ws);
    long long* d_cycles = reinterpret_cast<long long*>(ws + 256);
    unsigned long long* d_nanos = reinterpret_cast<unsigned long long*>(ws + 256 + 8192);
    unsigned* d_smid = reinterpret_cast<unsigned*>(ws + 256 + 2 * 8192);
    const int iters = 20000;
    k_mufu_rate<<<n_sm, 1024, 0, st>>>(200, -0.3f, sink, d_cycles, d_nanos, d_smid);   // warm-up
    MB_CUDA(cudaEventRecord(ev0, st));
    k_mufu_rate<<<n_sm, 1024, 0, st>>>(iters, -0.3f, sink, d_cycles, d_nanos, d_smid);
    MB_CUDA(cudaEventRecord(ev1, st));
    MB_CUDA(cudaGetLastError());
    MB_CUDA(cudaEventSynchronize(ev1));
    float ms = 0.f;
    MB_CUDA(cudaEventElapsedTime(&ms, ev0, ev1));
    static long long h_cycles[1024];
    static unsigned long long h_nanos[1024];
    static unsigned h_smid[1024];
    MB_CUDA(cudaMemcpy(h_cycles, d_cycles, sizeof(long long) * n_sm, cudaMemcpyDeviceToHost));
    MB_CUDA(cudaMemcpy(h_nanos, d_nanos, sizeof(unsigned long long) * n_sm, cudaMemcpyDeviceToHost));
    MB_CUDA(cudaMemcpy(h_smid, d_smid, sizeof(unsigned) * n_sm, cudaMemcpyDeviceToHost));
    {
        const double ops_block = 1024.0 * kChains * iters;
        double rate_sum = 0.0, mhz_sum = 0.0;
        bool seen[2048] = {false};
        bool one_per_sm = true;
        for (int b = 0; b < n_sm; ++b) {
            rate_sum += ops_block / (double)h_cycles[b];
            mhz_sum += (double)h_cycles[b] / (double)h_nanos[b] * 1e3;
            if (h_smid[b] >= 2048 || seen[h_smid[b]]) one_per_sm = false; else seen[h_smid[b]] = true;
        }
        r.sm_clock_mhz = mhz_sum / n_sm;
        r.mufu_ex2_per_s = ops_block * n_sm / (ms * 1e-3);
        // one block per SM: the block's own cycle count is the SM's; otherwise fall back to the device-wide rate and clock
        r.mufu_ex2_per_clk_per_sm = one_per_sm ? rate_sum / n_sm : r.mufu_ex2_per_s / ((double)n_sm * r.sm_clock_mhz * 1e6);
    }

    // ---- FP64 RED on random 256-byte rows ----
    double* table = reinterpret_cast<double*>(ws + (1 << 20));
    const size_t avail_rows = (device_bytes - (1 << 20)) / 256;
    auto red_rate = [&](size_t want_bytes, double* result) -> nd_status {
        size_t rows = 1;
        while (rows * 2 * 256 <= want_bytes && rows * 2 <= avail_rows) rows *= 2;
        *result = 0.0;
        if (rows * 256 < want_bytes / 2) return ND_OK;             // workspace too small for this case: reported as 0
        const int grid = n_sm * 8, it = 2000;
        MB_CUDA(cudaMemsetAsync(table, 0, rows * 256, st));
        k_red_rate<<<grid, 256, 0, st>>>(table, (unsigned)(rows - 1), 50);
        MB_CUDA(cudaEventRecord(ev0, st));
        k_red_rate<<<grid, 256, 0, st>>>(table, (unsigned)(rows - 1), it);
        MB_CUDA(cudaEventRecord(ev1, st));
        MB_CUDA(cudaGetLastError());
        MB_CUDA(cudaEventSynchronize(ev1));
        float t = 0.f;
        MB_CUDA(cudaEventElapsedTime(&t, ev0, ev1));
        *result = (double)grid * 256.0 * it / (t * 1e-3);
        return ND_OK;
    };
    nd_status rc = red_rate((size_t)32 << 20, &r.red_f64_l2_per_s);          // 32 MiB: inside the 126 MB L2
    if (rc == ND_OK) rc = red_rate((size_t)1 << 30, &r.red_f64_hbm_per_s);   // 1 GiB: 8 x L2
    cudaEventDestroy(ev0);
    cudaEventDestroy(ev1);
    if (rc != ND_OK) return rc;
    *out = r;
    return ND_OK;
}

// nd_setup.cuh -- the passes nd_problem_create makes over DEVICE-resident segment arrays (nd_problem_desc.seg_on_device):
// what the host loops of nd_problem_create do for host arrays, one thread per track (entry regions, SoA stream, A~_r) or
// per segment (validation).
#ifndef ND_SETUP_CUH
#define ND_SETUP_CUH
#include <cstdint>

#include "nd_kernels.cuh"

namespace ndk {

// flags[0] |= 1: a region id out of range; flags[0] |= 2: a length that is not finite and > 0
__global__ void __launch_bounds__(256) k_seg_validate(const int32_t* __restrict__ seg_region, const double* __restrict__ seg_length,
                                                      int64_t S, int R, int* flags)
{
    int bad = 0;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < S; k += (int64_t)gridDim.x * blockDim.x) {
        const int32_t r = seg_region[k];
        const double s = seg_length[k];
        if (r < 0 || r >= R) bad |= 1;
        if (!(s > 0.0) || !(s < 1.0e300)) bad |= 2;
    }
    bad = __reduce_or_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicOr(flags, bad);
}

// entry[2t] / entry[2t+1]: first region of the forward / backward chain of track t (-1: empty track).  Reads nothing when
// validation failed (the caller checks the flags first and launches this afterwards).
__global__ void __launch_bounds__(256) k_entry_regions(const int64_t* __restrict__ off, const int32_t* __restrict__ seg_region, int T,
                                                       int32_t* __restrict__ entry)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const int64_t k0 = off[t], k1 = off[t + 1];
    entry[2 * (size_t)t] = k1 > k0 ? seg_region[k0] : -1;
    entry[2 * (size_t)t + 1] = k1 > k0 ? seg_region[k1 - 1] : -1;
}

// the atomic kernel's SoA stream: every track run padded to a multiple of 4 with zero-length copies of its last segment
__global__ void __launch_bounds__(128) k_pack_soa(const int64_t* __restrict__ off, const int64_t* __restrict__ off_pad,
                                                  const int32_t* __restrict__ seg_region, const double* __restrict__ seg_length,
                                                  const int32_t* __restrict__ reg_mat, int T, uint32_t* __restrict__ seg_rm,
                                                  float* __restrict__ seg_len)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    int64_t at = off_pad[t];
    uint32_t last = 0;
    for (int64_t k = off[t]; k < off[t + 1]; ++k, ++at) {
        const int32_t r = seg_region[k];
        last = pack_rm((uint32_t)r, (uint32_t)reg_mat[r]);
        seg_rm[at] = last;
        seg_len[at] = (float)seg_length[k];
    }
    for (; at < off_pad[t + 1]; ++at) { seg_rm[at] = last; seg_len[at] = 0.f; }
}

// O-5: A~_r += 2 omega_a delta_a s (FP64 atomics)
__global__ void __launch_bounds__(128) k_track_volume(const int64_t* __restrict__ off, const int32_t* __restrict__ seg_region,
                                                      const double* __restrict__ seg_length, const double* __restrict__ w2, int T,
                                                      double* vol)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const double w = w2[t];
    for (int64_t k = off[t]; k < off[t + 1]; ++k) atomicAdd(vol + seg_region[k], w * seg_length[k]);
}

} // namespace ndk
#endif

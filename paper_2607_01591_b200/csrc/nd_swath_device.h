// nd_swath_device.h -- the swath/tile chunk stream built on the GPU from device-resident segments (nd_swath_device.cu).
#ifndef ND_SWATH_DEVICE_H
#define ND_SWATH_DEVICE_H
#include <cuda_runtime.h>

#include "nd_swath.h"

// DEVICE regions of the problem workspace the builder fills, with their capacities
struct NdSwathDeviceTargets {
    uint8_t* blob = nullptr;        size_t blob_cap = 0;        // bytes
    uint2* tile_ref = nullptr;      int64_t tile_cap = 0;       // entries (n_tiles + 1 are written)
    int64_t* swath_tile0 = nullptr; int64_t max_swaths = 0;     // [max_swaths + 1]
    int32_t* swath_track = nullptr;                             // [max_swaths][NT]
    int4* items = nullptr;                                      // [2 * max_swaths]
    uint16_t* slot_start = nullptr; size_t slot_start_cap = 0;  // bytes; only with prm.keep_slot_start
    void* scratch = nullptr;                                    // nd_swath_device_scratch_bytes(T, max_swaths)
    int lanes = 0;                                              // working threads per warp (0: default = 1)
};

size_t nd_swath_device_scratch_bytes(int64_t n_tracks, int64_t max_swaths);

// desc->seg_region / seg_length are DEVICE pointers, every other array of desc is on the host; d_region_material is the
// device copy of desc->region_material (already uploaded on `st`).  Fills the targets and the host-side meta data of *out
// (n_swaths, n_tiles, swath_track, swath_tile0, items, slot_start if requested, statistics, blob_bytes_device); out->blob and
// out->tile_ref stay empty.  Synchronises the stream.
nd_status nd_build_swaths_device(const nd_problem_desc* desc, const int32_t* d_region_material, const NdSwathParams& prm,
                                 const NdSwathDeviceTargets& tg, cudaStream_t st, NdSwathSet* out);

#endif

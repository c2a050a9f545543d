// nd_swath_device.cu -- SURVEY.md section 8(f) NEXT-1, second half: the swath/tile chunk stream of k_sweep_swath built ON
// THE GPU from device-resident segments (nd_tracks_generate_resident), so that no segment crosses PCIe in either direction.
//
// Which tracks share a swath is decided on the host from the track geometry (nd_swath_plan: O(T) work).  Cutting a swath
// into tiles and encoding its chunks is sequential along the swath, so one thread carries one swath through nd_swath_core
// -- the very function the host builder runs -- in two passes: COUNT (tiles and bytes per swath; the prefix sums are formed
// on the host, n_swaths numbers) and FILL.  The blobs of the two builders are equal byte for byte
// (tests/test_gpu_stream_device.py).  Only `lanes` threads of a warp work (default 1: swaths differ in length and in the
// path they take through the cutter, so the lanes of a warp would only serialise one another); the scratch of a swath
// (a few KB) lives in shared memory.
#include <algorithm>
#include <cstdio>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "nd.h"
#include "nd_internal.h"
#include "nd_swath.h"
#include "nd_swath_core.h"
#include "nd_swath_device.h"

namespace {

struct BuildParams {
    NdSwathCoreParams core;
    const int64_t* __restrict__ off;            // [T+1]
    const int32_t* __restrict__ seg_region;     // [S]
    const double* __restrict__ seg_length;      // [S]
    const int32_t* __restrict__ region_material;// [R]
    const int32_t* __restrict__ swath_track;    // [n_sw][NT]
    const double* __restrict__ lam0;            // [T]
    NdSwathCoreOut* counts;                     // [n_sw] (count pass: out)
    const int64_t* __restrict__ byte0;          // [n_sw] (fill pass)
    const int64_t* __restrict__ tile0;          // [n_sw+1] (fill pass)
    uint8_t* blob;
    uint32_t* tile_ref;                         // [n_tiles+1][2]
    uint16_t* slot_start;                       // [n_tiles][NT+1] or NULL
    int64_t n_sw;
    int lanes, scratch_bytes;
};

template <bool FILL>
__global__ void __launch_bounds__(128) k_swath_build(const BuildParams bp)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, warps = blockDim.x >> 5;
    if (lane >= bp.lanes) return;
    const int64_t sw = ((int64_t)blockIdx.x * warps + warp) * bp.lanes + lane;
    if (sw >= bp.n_sw) return;
    const NdSwathCoreParams& P = bp.core;
    const NdSwathScratch sc = nd_swath_scratch_at(smem + (size_t)(warp * bp.lanes + lane) * bp.scratch_bytes, P.NT, P.Kmax, P.Lmax);
    const int32_t* trk = bp.swath_track + sw * P.NT;
    NdSwathCoreOut o;
    if (FILL) {
        const int64_t b0 = bp.byte0[sw], t0 = bp.tile0[sw];
        nd_swath_core<true>(P, bp.off, bp.seg_region, bp.seg_length, bp.region_material, trk, bp.lam0, sc, bp.blob + b0,
                            bp.tile_ref + 2 * t0, (uint32_t)(b0 / 16), bp.slot_start ? bp.slot_start + t0 * (P.NT + 1) : nullptr, &o);
    } else {
        nd_swath_core<false>(P, bp.off, bp.seg_region, bp.seg_length, bp.region_material, trk, bp.lam0, sc, nullptr, nullptr, 0u, nullptr, &o);
        bp.counts[sw] = o;
    }
}

inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

} // namespace

size_t nd_swath_device_scratch_bytes(int64_t n_tracks, int64_t max_swaths)
{
    return up256(8 * (size_t)(n_tracks + 1)) + up256(8 * (size_t)n_tracks) + up256(sizeof(NdSwathCoreOut) * (size_t)max_swaths) +
           up256(8 * (size_t)max_swaths) + 256;
}

#define ND_SWD_CUDA(call)                                                                                \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            char buf_[512];                                                                              \
            snprintf(buf_, sizeof buf_, "%s failed: %s", #call, cudaGetErrorString(e_));                 \
            return nd_fail(ND_ERR_CUDA, buf_);                                                           \
        }                                                                                                \
    } while (0)

nd_status nd_build_swaths_device(const nd_problem_desc* desc, const int32_t* d_region_material, const NdSwathParams& prm,
                                 const NdSwathDeviceTargets& tg, cudaStream_t st, NdSwathSet* out)
{
    if (!desc->track_azim || !desc->track_ends)
        return nd_fail(ND_ERR_INVALID, "device-resident segments need the track geometry (track_azim, track_ends)");
    NdSwathCoreParams cp{};
    nd_status rc = nd_swath_check_params(desc, prm, &cp);
    if (rc != ND_OK) return rc;
    NdSwathPlan plan;
    rc = nd_swath_plan(desc, desc->track_azim, desc->track_ends, prm, &plan);
    if (rc != ND_OK) return rc;
    const int T = desc->n_tracks, NT = prm.NT;
    const int64_t n_sw = plan.n_swaths;
    if (n_sw > tg.max_swaths) return nd_fail(ND_ERR_WORKSPACE, "internal: more swaths than the workspace bound");
    cp.lag_len = nd_swath_lag_length(desc, desc->track_ends, prm.lag, 1);
    try {
        out->prm = prm;
        out->n_swaths = n_sw;
        out->swath_track = plan.swath_track;
        // scratch carve-up
        char* s = static_cast<char*>(tg.scratch);
        int64_t* d_off = reinterpret_cast<int64_t*>(s); s += up256(8 * (size_t)(T + 1));
        double* d_lam0 = reinterpret_cast<double*>(s); s += up256(8 * (size_t)T);
        NdSwathCoreOut* d_counts = reinterpret_cast<NdSwathCoreOut*>(s); s += up256(sizeof(NdSwathCoreOut) * (size_t)tg.max_swaths);
        int64_t* d_byte0 = reinterpret_cast<int64_t*>(s);
        ND_SWD_CUDA(cudaMemcpyAsync(d_off, desc->track_seg_offset, 8 * (size_t)(T + 1), cudaMemcpyHostToDevice, st));
        ND_SWD_CUDA(cudaMemcpyAsync(d_lam0, plan.lam0.data(), 8 * (size_t)T, cudaMemcpyHostToDevice, st));
        ND_SWD_CUDA(cudaMemcpyAsync(tg.swath_track, plan.swath_track.data(), 4 * plan.swath_track.size(), cudaMemcpyHostToDevice, st));
        BuildParams bp{};
        bp.core = cp; bp.off = d_off; bp.seg_region = desc->seg_region; bp.seg_length = desc->seg_length;
        bp.region_material = d_region_material; bp.swath_track = tg.swath_track; bp.lam0 = d_lam0; bp.counts = d_counts;
        bp.byte0 = d_byte0; bp.tile0 = tg.swath_tile0; bp.blob = tg.blob; bp.tile_ref = reinterpret_cast<uint32_t*>(tg.tile_ref);
        bp.slot_start = nullptr; bp.n_sw = n_sw;
        bp.lanes = tg.lanes > 0 && tg.lanes <= 32 ? tg.lanes : 1;
        bp.scratch_bytes = (int)nd_swath_scratch_bytes(NT, prm.Kmax, prm.Lmax);
        int warps = 4;
        while (warps > 1 && (size_t)warps * bp.lanes * bp.scratch_bytes > 160 * 1024) warps >>= 1;
        const size_t smem = (size_t)warps * bp.lanes * bp.scratch_bytes;
        if (smem > 200 * 1024) return nd_fail(ND_ERR_INVALID, "swath parameters: the cutter's scratch exceeds shared memory");
        ND_SWD_CUDA(cudaFuncSetAttribute(k_swath_build<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ND_SWD_CUDA(cudaFuncSetAttribute(k_swath_build<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        const int64_t per_block = (int64_t)warps * bp.lanes;
        const unsigned grid = (unsigned)((n_sw + per_block - 1) / per_block);
        // ---- COUNT ----
        std::vector<NdSwathCoreOut> h_counts((size_t)n_sw);
        if (n_sw > 0) {
            k_swath_build<false><<<grid, 32 * warps, smem, st>>>(bp);
            ND_SWD_CUDA(cudaGetLastError());
            ND_SWD_CUDA(cudaMemcpyAsync(h_counts.data(), d_counts, sizeof(NdSwathCoreOut) * (size_t)n_sw, cudaMemcpyDeviceToHost, st));
        }
        ND_SWD_CUDA(cudaStreamSynchronize(st));
        out->swath_tile0.assign((size_t)n_sw + 1, 0);
        std::vector<int64_t> byte0((size_t)n_sw + 1, 0), cost((size_t)n_sw);
        int64_t sum_regions = 0, sum_seg = 0, sum_slots = 0;
        int max_head = 0, max_rec = 0;
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            const NdSwathCoreOut& c = h_counts[(size_t)sw];
            out->swath_tile0[sw + 1] = out->swath_tile0[sw] + c.n_tiles;
            byte0[sw + 1] = byte0[sw] + c.n_bytes;
            sum_regions += c.sum_regions; sum_seg += c.n_seg; sum_slots += c.sum_max_cnt * c.n_active;
            max_head = std::max(max_head, c.max_head); max_rec = std::max(max_rec, c.max_rec);
            cost[(size_t)sw] = c.sum_max_cnt;
        }
        out->n_tiles = out->swath_tile0[n_sw];
        const size_t total = (size_t)byte0[n_sw];
        if (total / 16 >= 0xffffffffull) return nd_fail(ND_ERR_RANGE, "swath stream exceeds 64 GiB");
        if (total > tg.blob_cap || out->n_tiles + 1 > tg.tile_cap)
            return nd_fail(ND_ERR_WORKSPACE, "internal: swath stream larger than its workspace bound");
        const bool keep = prm.keep_slot_start;
        if (keep && (!tg.slot_start || (size_t)out->n_tiles * (NT + 1) * 2 > tg.slot_start_cap))
            return nd_fail(ND_ERR_WORKSPACE, "internal: slot_start larger than its workspace bound");
        out->blob_bytes_device = total;
        // ---- FILL ----
        ND_SWD_CUDA(cudaMemcpyAsync(tg.swath_tile0, out->swath_tile0.data(), 8 * (size_t)(n_sw + 1), cudaMemcpyHostToDevice, st));
        ND_SWD_CUDA(cudaMemcpyAsync(d_byte0, byte0.data(), 8 * (size_t)n_sw, cudaMemcpyHostToDevice, st));
        ND_SWD_CUDA(cudaMemsetAsync(tg.blob, 0, total, st));   // padding bytes of the chunks stay zero
        const uint2 sentinel = make_uint2((uint32_t)(total / 16), 0u);   // chunk k spans [k, k+1)
        ND_SWD_CUDA(cudaMemcpyAsync(tg.tile_ref + out->n_tiles, &sentinel, sizeof sentinel, cudaMemcpyHostToDevice, st));
        bp.slot_start = keep ? tg.slot_start : nullptr;
        if (n_sw > 0) {
            k_swath_build<true><<<grid, 32 * warps, smem, st>>>(bp);
            ND_SWD_CUDA(cudaGetLastError());
        }
        out->slot_start.clear();
        if (keep) {
            out->slot_start.resize((size_t)out->n_tiles * (NT + 1));
            ND_SWD_CUDA(cudaMemcpyAsync(out->slot_start.data(), tg.slot_start, 2 * out->slot_start.size(), cudaMemcpyDeviceToHost, st));
        }
        nd_swath_items(plan, cost.data(), prm.item_order, &out->items);
        static_assert(sizeof(NdSwathItem) == sizeof(int4), "work item layout");
        ND_SWD_CUDA(cudaMemcpyAsync(tg.items, out->items.data(), sizeof(NdSwathItem) * out->items.size(), cudaMemcpyHostToDevice, st));
        ND_SWD_CUDA(cudaStreamSynchronize(st));
        out->max_head_bytes = max_head;
        out->max_rec_bytes = max_rec;
        out->mean_regions_per_tile = out->n_tiles ? (double)sum_regions / (double)out->n_tiles : 0.0;
        out->mean_segments_per_tile = out->n_tiles ? (double)sum_seg / (double)out->n_tiles : 0.0;
        out->lockstep_efficiency = sum_slots ? (double)sum_seg / (double)sum_slots : 1.0;
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_build_swaths_device: out of host memory");
    }
    return ND_OK;
}

// nd_swath.h -- host-side construction of the swath/tile chunk stream of k_sweep_swath (row A1 of DESIGN.md).
//
// Tracks of one angle are sorted by their perpendicular coordinate and grouped into SWATHS of NT adjacent tracks;
// one thread block carries a swath, one lane group ("slot") per track, so the angular flux of a track stays in
// registers from one end of the track to the other.  A swath is cut along the track direction into TILES: the
// tracks advance either by equal counts (every track Kmax segments) or, when their fronts have drifted apart, in
// geometric lock step (always the track whose front is furthest behind) until one of them has Kmax segments in the
// tile; in both modes a tile touches at most Lmax distinct regions.  A tile is one contiguous, 16-byte aligned
// CHUNK made of a HEAD and a RECORD part, each fetched by one bulk (TMA) copy into its own shared-memory ring:
//   head  u32 hdr[4]          L | nseg << 16 ;  off_regions (16-byte units from the chunk start) ;  head bytes ;  chunk bytes
//         u16 slot_start[NT+1] per-track prefix into rec[]                                     (padded to 16 B)
//         u32 regions[L][2]    { global region id (q row to stage, tally row to flush) ;
//                                first delta-buffer row | one past the last << 16 }             (padded to 16 B),
//                              in descending order of their row counts
//   rec   rec[nseg]            16 bytes each: { f32 length ; u32 q-row byte offset ; u32 Sigma_t-row byte offset ;
//                              u32 delta-row byte offset }, slot-major, forward order; the backward direction walks
//                              the same records in reverse
// Delta rows are REGION-MAJOR: the rows of a region are consecutive, ordered by slot then by position along
// the track, so the flush adds up a contiguous run of rows per region (no index list) and adjacent tracks crossing
// the same region store into adjacent rows.  A segment's weighted flux change is simply STORED in its own row (a
// track may re-enter a region; every visit has its own row).
#ifndef ND_SWATH_H
#define ND_SWATH_H
#include <cstddef>
#include <cstdint>
#include <memory>
#include <vector>

#include "nd.h"

struct NdSwathParams {
    int NT;       // tracks per swath = slots per thread block
    int Kmax;     // max segments of one track in a tile
    int Lmax;     // max distinct regions in a tile
    int NC;       // slots whose Sigma_t rows share one shared-memory line (bank-conflict-free layout for narrow rows)
    int row_bytes;// bytes of one (region, all groups) FP32 row = 4 * Gs
    double lag;   // >= 0: while the fronts of the swath's tracks lie within `lag` mean segment lengths of each other a
                  // tile gives EVERY track Kmax segments (no idle slot steps); beyond it the tile is cut geometrically
                  // (the track furthest behind advances first) until the fronts are level again.  < 0: always geometric.
    int NCq = 0;  // copies of a q row per shared line (0: = NC).  1 = one copy per region: adjacent slots in the same region
                  // read it as a broadcast, slots in different regions may meet in a bank
    bool keep_slot_start = false;   // also return every tile's slot_start array on the host (the CMFD crossing lists need it)
    int item_order = 0;   // 0: work items most expensive first (load balance); 1: angle by angle, adjacent swaths
                          // consecutively, forward then backward (blocks that run together touch neighbouring regions)
};

struct NdSwathItem { int32_t swath, dir, cost, reserved; };
struct NdSwathTileRef { uint32_t off16, head16; };   // chunk offset and head size, both in 16-byte units

// Byte buffer that is NOT value-initialised: the chunk stream of a 5e8-segment problem (8-9 GB) is written exactly once by
// parallel copies; zero-filling it first (std::vector::resize) cost seconds of single-threaded page faults.
struct NdRawBytes {
    std::unique_ptr<uint8_t[]> p;
    size_t n = 0;
    void resize_uninitialised(size_t bytes) { p.reset(bytes ? new uint8_t[bytes] : nullptr); n = bytes; }
    uint8_t* data() { return p.get(); }
    const uint8_t* data() const { return p.get(); }
    size_t size() const { return n; }
};

struct NdSwathSet {
    NdSwathParams prm{};
    int64_t n_swaths = 0, n_tiles = 0;
    std::vector<int32_t> swath_track;     // [n_swaths][NT] canonical track id or -1
    std::vector<int64_t> swath_tile0;     // [n_swaths+1] prefix into tile_ref
    std::vector<NdSwathTileRef> tile_ref; // [n_tiles+1] (+ end sentinel: chunk k spans [off16[k], off16[k+1]))
    std::vector<NdSwathItem> items;       // work items (swath, direction)
    std::vector<uint16_t> slot_start;     // [n_tiles][NT+1] (only with prm.keep_slot_start)
    NdRawBytes blob;                      // all chunks (every byte written by nd_build_swaths)
    size_t blob_bytes_device = 0;         // device builder: bytes of the stream it wrote into the workspace (blob stays empty)
    int max_head_bytes = 0, max_rec_bytes = 0;
    double mean_regions_per_tile = 0.0, mean_segments_per_tile = 0.0, lockstep_efficiency = 0.0;
};

inline int nd_swath_pad16(int x) { return (x + 15) / 16 * 16; }

// largest head / record part the parameters allow (the kernel's staging rings have these sizes)
inline int nd_swath_head_capacity(const NdSwathParams& p)
{
    return 16 + nd_swath_pad16(2 * (p.NT + 1)) + nd_swath_pad16(8 * p.Lmax);
}
inline int nd_swath_rec_capacity(const NdSwathParams& p) { return 16 * p.NT * p.Kmax; }

// upper bounds used to size the device workspace before the stream is built
inline int64_t nd_swath_max_tiles(const NdSwathParams& p, int64_t n_segments, int64_t n_tracks)
{
    const int m = p.Kmax < p.Lmax ? p.Kmax : p.Lmax;
    return n_segments / m + n_tracks + 2;
}
inline size_t nd_swath_max_blob(const NdSwathParams& p, int64_t n_segments, int64_t n_tracks)
{
    // head: 16 + slot prefix + 8 bytes per region (<= one region per segment) + two paddings
    const size_t per_tile = 16 + (size_t)nd_swath_pad16(2 * (p.NT + 1)) + 2 * 16;
    return (size_t)nd_swath_max_tiles(p, n_segments, n_tracks) * per_tile + 24 * (size_t)n_segments + 256;
}

struct NdSwathCoreParams;

// which tracks share a swath (needs the track geometry, no segment)
struct NdSwathPlan {
    int64_t n_swaths = 0;
    std::vector<int32_t> swath_track;   // [n_swaths][NT] canonical track id or -1
    std::vector<int32_t> group;         // [n_swaths] angle id of the swath's tracks
    std::vector<double> lam0;           // [T] coordinate of every track's start point along its angle's direction
};

nd_status nd_swath_check_params(const nd_problem_desc* desc, const NdSwathParams& prm, NdSwathCoreParams* core);
nd_status nd_swath_plan(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends, const NdSwathParams& prm,
                        NdSwathPlan* plan);
void nd_swath_items(const NdSwathPlan& plan, const int64_t* cost, int item_order, std::vector<NdSwathItem>* items);
double nd_swath_lag_length(const nd_problem_desc* desc, const double* track_ends, double lag, int n_threads);

// track_azim / track_ends may be NULL (no geometry): tracks are then grouped in descriptor order.
nd_status nd_build_swaths(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends,
                          const NdSwathParams& prm, int n_threads, NdSwathSet* out);

#endif

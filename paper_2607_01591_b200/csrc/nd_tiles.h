// nd_tiles.h -- host-side construction of the swath/tile chunk stream used by k_sweep_private (row A1).
//
// Tracks of one angle are sorted by their perpendicular coordinate and grouped into SWATHS of B adjacent
// tracks.  A swath is cut along the track direction into TILES: maximal runs (in along-track coordinate) whose
// segments touch at most Lw distinct regions and number at most Nmax.  A tile is stored as one contiguous,
// 16-byte aligned CHUNK:
//     u32 L            number of distinct regions (<= Lw)
//     u32 bytes        chunk size, multiple of 16
//     u32 nseg         segments in the chunk
//     u32 reserved
//     u16 seg_start[B+1]   (padded to 16 B)  per-track prefix into the segment arrays
//     u32 regions[pad4(L)]                   region | material << 24
//     f32 len[pad4(nseg)]                    track-major, forward order
//     u16 im[pad8(nseg)]                     local region index | material << 8
// The kernel stages a chunk into shared memory with one bulk copy and then only touches shared memory in its
// segment loop; the backward direction reads the same chunks in reverse.
#ifndef ND_TILES_H
#define ND_TILES_H
#include <cstdint>
#include <vector>

#include "nd.h"

struct NdTileParams {
    int B;        // tracks per swath
    int Lw;       // regions per private window (<= 255, >= B)
    int Nmax;     // max segments per chunk
    int TPW;      // swaths per work item (track slots per warp)
};

struct NdTileItem { int32_t first_swath, n_swaths, dir, cost; };

struct NdTileSet {
    NdTileParams prm{};
    int64_t n_swaths = 0, n_tiles = 0;
    std::vector<int32_t> swath_track;     // [n_swaths][B] canonical track id or -1
    std::vector<int64_t> swath_tile0;     // [n_swaths+1] prefix into tile_chunk
    std::vector<uint32_t> tile_chunk;     // [n_tiles] chunk offset in 16-byte units
    std::vector<NdTileItem> items;        // work items, most expensive first
    std::vector<uint8_t> blob;            // all chunks
    int max_chunk_bytes = 0;
    double mean_regions_per_tile = 0.0, mean_segments_per_tile = 0.0;
};

inline int nd_chunk_capacity_bytes(const NdTileParams& p)
{
    auto pad = [](int x, int a) { return (x + a - 1) / a * a; };
    return 16 + pad(2 * (p.B + 1), 16) + 4 * pad(p.Lw, 4) + 4 * pad(p.Nmax, 4) + 2 * pad(p.Nmax, 8);
}

// track_azim / track_ends may be NULL (no geometry): tracks are then grouped in descriptor order.
nd_status nd_build_tiles(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends,
                         const NdTileParams& prm, int n_threads, NdTileSet* out);

#endif

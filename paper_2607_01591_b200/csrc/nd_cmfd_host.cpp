// nd_cmfd_host.cpp -- host-side geometry of the CMFD step (C-1 / C-2):
// which pairs of coarse cells the tracks join.  Integer work only; the arithmetic of the method runs in CUDA kernels.
#include <algorithm>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "nd_internal.h"

// C-2: the interior surfaces of the coarse mesh are the unordered cell pairs (lo < hi) that
//   (a) two consecutive segments of some track join, or
//   (b) a reflective hand-over joins: the cell in which chain (t, d) ends and the cell in which the chain it links to
//       begins (they differ when two cyclic tracks meet at a mesh vertex on the boundary).
// Output sorted by (lo, hi).
extern "C" nd_status nd_cmfd_surfaces(const nd_problem_desc* desc, int32_t n_cells, const int32_t* cell, int32_t capacity,
                                      int32_t* n_pairs_out, int32_t* pair_lo, int32_t* pair_hi)
{
    if (!desc || !cell || !n_pairs_out) return nd_fail(ND_ERR_NULL, "nd_cmfd_surfaces: NULL argument");
    if (!desc->track_seg_offset || !desc->seg_region || !desc->link) return nd_fail(ND_ERR_NULL, "nd_cmfd_surfaces: a descriptor array is NULL");
    if (n_cells < 1 || desc->n_regions < 1 || desc->n_tracks < 1 || capacity < 0)
        return nd_fail(ND_ERR_INVALID, "nd_cmfd_surfaces: n_cells, n_regions, n_tracks must be >= 1 and capacity >= 0");
    if (capacity > 0 && (!pair_lo || !pair_hi)) return nd_fail(ND_ERR_NULL, "nd_cmfd_surfaces: pair_lo / pair_hi are NULL");
    const int32_t R = desc->n_regions, T = desc->n_tracks;
    const int64_t* off = desc->track_seg_offset;
    for (int32_t r = 0; r < R; ++r)
        if (cell[r] < 0 || cell[r] >= n_cells) return nd_fail(ND_ERR_RANGE, "nd_cmfd_surfaces: cell[r] out of [0, n_cells)");
    if (off[0] != 0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_surfaces: track_seg_offset[0] must be 0");
    for (int32_t t = 0; t < T; ++t)
        if (off[t + 1] < off[t]) return nd_fail(ND_ERR_INVALID, "nd_cmfd_surfaces: track_seg_offset must be non-decreasing");
    const int64_t S = off[T];
    for (int64_t k = 0; k < S; ++k)
        if (desc->seg_region[k] < 0 || desc->seg_region[k] >= R) return nd_fail(ND_ERR_RANGE, "nd_cmfd_surfaces: seg_region out of range");
    for (int64_t e = 0; e < 2 * (int64_t)T; ++e)
        if (desc->link[e] < -1 || desc->link[e] >= 2 * T) return nd_fail(ND_ERR_RANGE, "nd_cmfd_surfaces: link out of range");
    std::vector<int64_t> keys;
    try {
        auto key_of = [n_cells](int32_t a, int32_t b) { return (int64_t)std::min(a, b) * n_cells + std::max(a, b); };
#pragma omp parallel
        {
            std::vector<int64_t> mine;
            int64_t last_key = -1;   // consecutive crossings of adjacent tracks repeat the same pair: skip the obvious duplicates
#pragma omp for schedule(static) nowait
            for (int32_t t = 0; t < T; ++t) {
                const int64_t k0 = off[t], k1 = off[t + 1];
                for (int64_t k = k0 + 1; k < k1; ++k) {
                    const int32_t a = cell[desc->seg_region[k - 1]], b = cell[desc->seg_region[k]];
                    if (a != b) {
                        const int64_t key = key_of(a, b);
                        if (key != last_key) { mine.push_back(key); last_key = key; }
                    }
                }
                if (k1 > k0)
                    for (int d = 0; d < 2; ++d) {                     // chain (t, d) ends in the last (d = 0) / first (d = 1) region
                        const int32_t lk = desc->link[2 * (int64_t)t + d];
                        if (lk < 0) continue;
                        const int32_t t2 = lk >> 1, d2 = lk & 1;
                        if (off[t2 + 1] <= off[t2]) continue;         // the receiving track has no segment
                        const int32_t a = cell[desc->seg_region[d == 0 ? k1 - 1 : k0]];
                        const int32_t b = cell[desc->seg_region[d2 == 0 ? off[t2] : off[t2 + 1] - 1]];
                        if (a != b) mine.push_back(key_of(a, b));
                    }
            }
            std::sort(mine.begin(), mine.end());
            mine.erase(std::unique(mine.begin(), mine.end()), mine.end());
#pragma omp critical
            keys.insert(keys.end(), mine.begin(), mine.end());
        }
        std::sort(keys.begin(), keys.end());
        keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_cmfd_surfaces: out of host memory");
    }
    if (keys.size() > (size_t)INT32_MAX) return nd_fail(ND_ERR_RANGE, "nd_cmfd_surfaces: more than 2^31 surfaces");
    *n_pairs_out = (int32_t)keys.size();
    if (capacity == 0) return ND_OK;                                  // size query
    if ((size_t)capacity < keys.size()) return nd_fail(ND_ERR_INVALID, "nd_cmfd_surfaces: capacity smaller than the number of surfaces");
    for (size_t i = 0; i < keys.size(); ++i) {
        pair_lo[i] = (int32_t)(keys[i] / n_cells);
        pair_hi[i] = (int32_t)(keys[i] % n_cells);
    }
    return ND_OK;
}

// nd_tiles.cpp -- builds the swath/tile chunk stream (see nd_tiles.h).  Host code, OpenMP over swaths.
// Geometry is used only to ORDER work (which tracks share a swath, where tiles are cut); every segment of the
// descriptor is assigned to exactly one chunk whatever the geometry says, so results never depend on it.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <numeric>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "nd_internal.h"
#include "nd_tiles.h"

namespace {

inline int pad_to(int x, int a) { return (x + a - 1) / a * a; }

struct SwathBuild {
    std::vector<uint8_t> bytes;        // this swath's chunks, concatenated
    std::vector<uint32_t> chunk_rel;   // chunk offsets relative to the swath's first byte, 16-B units
    int64_t n_seg = 0;
    int64_t sum_regions = 0;
    int max_chunk = 0;
};

} // namespace

nd_status nd_build_tiles(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends,
                         const NdTileParams& prm, int n_threads, NdTileSet* out)
{
    const int T = desc->n_tracks, R = desc->n_regions, B = prm.B, Lw = prm.Lw, Nmax = prm.Nmax;
    if (B < 1 || B > 64 || Lw < B || Lw > 255 || Nmax < B || Nmax > 4096 || prm.TPW < 1)
        return nd_fail(ND_ERR_INVALID, "tile parameters: need 1 <= B <= 64, B <= Lw <= 255, B <= Nmax <= 4096");
    try {
        out->prm = prm;
        // ---- 1. order tracks: by angle id, then by perpendicular coordinate ----
        std::vector<int32_t> order(T);
        std::iota(order.begin(), order.end(), 0);
        std::vector<double> perp(T, 0.0), lam0(T, 0.0);
        std::vector<int32_t> group(T, 0);
        if (track_azim && track_ends) {
            // direction of a group = direction of its first track
            int32_t gmax = 0;
            for (int t = 0; t < T; ++t) { group[t] = track_azim[t]; if (group[t] < 0) group[t] = 0; gmax = std::max(gmax, group[t]); }
            std::vector<double> ux((size_t)gmax + 1, 0.0), uy((size_t)gmax + 1, 0.0);
            std::vector<char> have((size_t)gmax + 1, 0);
            for (int t = 0; t < T; ++t) {
                const int g = group[t];
                if (have[g]) continue;
                const double dx = track_ends[4 * (size_t)t + 2] - track_ends[4 * (size_t)t];
                const double dy = track_ends[4 * (size_t)t + 3] - track_ends[4 * (size_t)t + 1];
                const double h = std::sqrt(dx * dx + dy * dy);
                if (h > 0.0 && std::isfinite(h)) { ux[g] = dx / h; uy[g] = dy / h; have[g] = 1; }
            }
            for (int t = 0; t < T; ++t) {
                const int g = group[t];
                const double x0 = track_ends[4 * (size_t)t], y0 = track_ends[4 * (size_t)t + 1];
                perp[t] = x0 * uy[g] - y0 * ux[g];
                lam0[t] = x0 * ux[g] + y0 * uy[g];
                if (!std::isfinite(perp[t])) perp[t] = 0.0;
                if (!std::isfinite(lam0[t])) lam0[t] = 0.0;
            }
            std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
                if (group[a] != group[b]) return group[a] < group[b];
                return perp[a] < perp[b];
            });
        }
        // ---- 2. swaths: B consecutive tracks of one group ----
        std::vector<int32_t>& st = out->swath_track;
        st.clear();
        std::vector<int32_t> swath_group;
        for (int i = 0; i < T;) {
            int n = 0;
            const int g = group[order[i]];
            while (n < B && i + n < T && group[order[i + n]] == g) ++n;
            for (int b = 0; b < B; ++b) st.push_back(b < n ? order[i + b] : -1);
            swath_group.push_back(g);
            i += n;
        }
        const int64_t n_sw = (int64_t)swath_group.size();
        out->n_swaths = n_sw;
        // ---- 3. cut every swath into tiles and encode the chunks ----
        std::vector<SwathBuild> built((size_t)n_sw);
#ifdef _OPENMP
        const int nth = n_threads > 0 ? n_threads : omp_get_max_threads();
#else
        const int nth = 1;
        (void)n_threads;
#endif
        const int64_t* off = desc->track_seg_offset;
#pragma omp parallel num_threads(nth)
        {
            std::vector<int32_t> stamp((size_t)R, -1), lidx((size_t)R, 0);
            int32_t tile_serial = 0;
            std::vector<int64_t> cur(B), first(B), endk(B);
            std::vector<double> lam(B);
            std::vector<uint32_t> regions;
            regions.reserve(Lw);
#pragma omp for schedule(dynamic, 8)
            for (int64_t sw = 0; sw < n_sw; ++sw) {
                SwathBuild& sb = built[(size_t)sw];
                const int32_t* trk = &st[(size_t)sw * B];
                int64_t remaining = 0;
                for (int b = 0; b < B; ++b) {
                    if (trk[b] >= 0) { cur[b] = off[trk[b]]; endk[b] = off[trk[b] + 1]; lam[b] = lam0[trk[b]]; }
                    else { cur[b] = endk[b] = 0; lam[b] = 0.0; }
                    remaining += endk[b] - cur[b];
                }
                sb.n_seg = remaining;
                do { // at least one (possibly empty) tile per swath
                    if (++tile_serial == INT32_MAX) { std::fill(stamp.begin(), stamp.end(), -1); tile_serial = 0; }
                    regions.clear();
                    for (int b = 0; b < B; ++b) first[b] = cur[b];
                    int nseg = 0;
                    while (remaining > 0 && nseg < Nmax) {
                        int bs = -1;
                        for (int b = 0; b < B; ++b)
                            if (cur[b] < endk[b] && (bs < 0 || lam[b] < lam[bs])) bs = b;
                        const int64_t k = cur[bs];
                        const int32_t r = desc->seg_region[k];
                        if (stamp[r] != tile_serial) {
                            if ((int)regions.size() == Lw) break;
                            stamp[r] = tile_serial;
                            lidx[r] = (int32_t)regions.size();
                            regions.push_back((uint32_t)r | ((uint32_t)desc->region_material[r] << 24));
                        }
                        lam[bs] += desc->seg_length[k];
                        ++cur[bs]; ++nseg; --remaining;
                    }
                    // encode
                    const int L = (int)regions.size();
                    const int h0 = 16, h1 = h0 + pad_to(2 * (B + 1), 16), h2 = h1 + 4 * pad_to(L, 4), h3 = h2 + 4 * pad_to(nseg, 4);
                    const int bytes = h3 + pad_to(2 * pad_to(nseg, 8), 16);
                    const size_t base = sb.bytes.size();
                    sb.chunk_rel.push_back((uint32_t)(base / 16));
                    sb.bytes.resize(base + (size_t)bytes, 0);
                    uint8_t* c = sb.bytes.data() + base;
                    uint32_t hdr[4] = {(uint32_t)L, (uint32_t)bytes, (uint32_t)nseg, 0u};
                    memcpy(c, hdr, 16);
                    uint16_t* ss = reinterpret_cast<uint16_t*>(c + h0);
                    uint32_t* rg = reinterpret_cast<uint32_t*>(c + h1);
                    float* ln = reinterpret_cast<float*>(c + h2);
                    uint16_t* im = reinterpret_cast<uint16_t*>(c + h3);
                    for (int l = 0; l < L; ++l) rg[l] = regions[l];
                    int o = 0;
                    for (int b = 0; b < B; ++b) {
                        ss[b] = (uint16_t)o;
                        for (int64_t k = first[b]; k < cur[b]; ++k, ++o) {
                            const int32_t r = desc->seg_region[k];
                            ln[o] = (float)desc->seg_length[k];
                            im[o] = (uint16_t)(lidx[r] | (desc->region_material[r] << 8));
                        }
                    }
                    ss[B] = (uint16_t)o;
                    sb.sum_regions += L;
                    sb.max_chunk = std::max(sb.max_chunk, bytes);
                } while (remaining > 0);
            }
        }
        // ---- 4. concatenate ----
        out->swath_tile0.assign((size_t)n_sw + 1, 0);
        std::vector<size_t> byte0((size_t)n_sw + 1, 0);
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            out->swath_tile0[sw + 1] = out->swath_tile0[sw] + (int64_t)built[sw].chunk_rel.size();
            byte0[sw + 1] = byte0[sw] + built[sw].bytes.size();
        }
        out->n_tiles = out->swath_tile0[n_sw];
        if (byte0[n_sw] / 16 >= 0xffffffffull) return nd_fail(ND_ERR_RANGE, "tile stream exceeds 64 GiB");
        out->tile_chunk.resize((size_t)out->n_tiles + 1);
        out->tile_chunk[(size_t)out->n_tiles] = (uint32_t)(byte0[n_sw] / 16);   // end sentinel: chunk k spans [k, k+1)
        out->blob.resize(byte0[n_sw]);
        int64_t sum_regions = 0, sum_seg = 0;
        int max_chunk = 0;
        for (int64_t sw = 0; sw < n_sw; ++sw) { sum_regions += built[sw].sum_regions; sum_seg += built[sw].n_seg; max_chunk = std::max(max_chunk, built[sw].max_chunk); }
#pragma omp parallel for schedule(dynamic, 64) num_threads(nth)
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            SwathBuild& sb = built[(size_t)sw];
            if (!sb.bytes.empty()) memcpy(out->blob.data() + byte0[sw], sb.bytes.data(), sb.bytes.size());
            const uint32_t b16 = (uint32_t)(byte0[sw] / 16);
            for (size_t i = 0; i < sb.chunk_rel.size(); ++i) out->tile_chunk[(size_t)out->swath_tile0[sw] + i] = b16 + sb.chunk_rel[i];
            std::vector<uint8_t>().swap(sb.bytes);
        }
        out->max_chunk_bytes = max_chunk;
        out->mean_regions_per_tile = out->n_tiles ? (double)sum_regions / (double)out->n_tiles : 0.0;
        out->mean_segments_per_tile = out->n_tiles ? (double)sum_seg / (double)out->n_tiles : 0.0;
        // ---- 5. work items: TPW consecutive swaths of one group, both directions, most expensive first ----
        out->items.clear();
        for (int64_t s0 = 0; s0 < n_sw;) {
            int n = 0;
            int64_t cost = 0;
            while (n < prm.TPW && s0 + n < n_sw && swath_group[s0 + n] == swath_group[s0]) { cost = std::max<int64_t>(cost, built[s0 + n].n_seg); ++n; }
            const int32_t c32 = (int32_t)std::min<int64_t>(cost, INT32_MAX);
            out->items.push_back({(int32_t)s0, n, 0, c32});
            out->items.push_back({(int32_t)s0, n, 1, c32});
            s0 += n;
        }
        std::stable_sort(out->items.begin(), out->items.end(), [](const NdTileItem& a, const NdTileItem& b) { return a.cost > b.cost; });
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_build_tiles: out of host memory");
    }
    return ND_OK;
}

// nd_swath.cpp -- builds the swath/tile chunk stream (see nd_swath.h).  Host code, OpenMP over swaths.
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
#include "nd_swath.h"

namespace {

struct SwathBuild {
    std::vector<uint8_t> bytes;        // this swath's chunks, concatenated
    std::vector<uint32_t> chunk_rel;   // chunk offsets relative to the swath's first byte, 16-B units
    std::vector<uint32_t> head16;      // head size of every chunk, 16-B units
    std::vector<uint16_t> slot_start;  // [tiles][NT+1] when requested
    int64_t n_seg = 0, sum_regions = 0, sum_max_cnt = 0, n_active = 0;
    int max_head = 0, max_rec = 0;
    int32_t group = 0;                 // angle id of the swath's tracks
    double perp = 0.0;                 // perpendicular coordinate of its first track
};

} // namespace

nd_status nd_build_swaths(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends,
                          const NdSwathParams& prm, int n_threads, NdSwathSet* out)
{
    const int T = desc->n_tracks, R = desc->n_regions, NT = prm.NT, Kmax = prm.Kmax, Lmax = prm.Lmax, NC = prm.NC;
    if (NT < 1 || NT > 1024 || Kmax < 1 || Lmax < 1 || NC < 1 || NT % NC != 0 || prm.row_bytes < 16 || prm.row_bytes % 16 != 0)
        return nd_fail(ND_ERR_INVALID, "swath parameters out of range");
    const int64_t line = (int64_t)NC * prm.row_bytes;   // bytes between consecutive sigma_t rows in shared memory
    const int NCq = prm.NCq > 0 ? prm.NCq : NC;
    const int64_t line_q = (int64_t)NCq * prm.row_bytes; // bytes between consecutive q rows
    const int64_t row_bytes = prm.row_bytes;             // bytes between consecutive delta rows
    if (Lmax > 65535 || (int64_t)NT * Kmax > 65535 || nd_swath_head_capacity(prm) / 16 > 65535 ||
        (int64_t)Lmax * line_q > (1ll << 30) || (int64_t)desc->n_materials * line > (1ll << 30))
        return nd_fail(ND_ERR_INVALID, "swath parameters: tile sizes must fit 16 bits");
    try {
        out->prm = prm;
        // ---- 1. order tracks: by angle id, then by perpendicular coordinate ----
        std::vector<int32_t> order(T);
        std::iota(order.begin(), order.end(), 0);
        std::vector<double> lam0(T, 0.0), perp(T, 0.0);
        std::vector<int32_t> group(T, 0);
        if (track_azim && track_ends) {
            int32_t gmax = 0;
            for (int t = 0; t < T; ++t) { group[t] = track_azim[t] < 0 ? 0 : track_azim[t]; gmax = std::max(gmax, group[t]); }
            std::vector<double> ux((size_t)gmax + 1, 0.0), uy((size_t)gmax + 1, 0.0);
            std::vector<char> have((size_t)gmax + 1, 0);
            for (int t = 0; t < T; ++t) {   // direction of a group = direction of its first non-degenerate track
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
        // ---- 2. swaths: NT consecutive tracks of one group ----
        std::vector<int32_t>& st = out->swath_track;
        st.clear();
        for (int i = 0; i < T;) {
            int n = 0;
            const int g = group[order[i]];
            while (n < NT && i + n < T && group[order[i + n]] == g) ++n;
            for (int b = 0; b < NT; ++b) st.push_back(b < n ? order[i + b] : -1);
            i += n;
        }
        const int64_t n_sw = (int64_t)(st.size() / NT);
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
        double lag_len = -1.0;
        if (prm.lag >= 0.0) {
            double sum = 0.0;
            const int64_t S = off[T];
#pragma omp parallel for reduction(+ : sum) num_threads(nth)
            for (int64_t k = 0; k < S; ++k) sum += desc->seg_length[k];
            lag_len = S > 0 ? prm.lag * sum / (double)S : 0.0;
        }
#pragma omp parallel num_threads(nth)
        {
            std::vector<int32_t> stamp((size_t)R, -1), lidx((size_t)R, 0);
            int32_t tile_serial = 0;
            std::vector<int64_t> cur(NT), first(NT), endk(NT);
            std::vector<double> lam(NT);
            std::vector<int> cnt(NT);
            std::vector<uint32_t> regions;
            std::vector<int> rcount, rfill, perm, sorted_count;
            std::vector<uint32_t> sorted_regions;
            regions.reserve(Lmax);
#pragma omp for schedule(dynamic, 4)
            for (int64_t sw = 0; sw < n_sw; ++sw) {
                SwathBuild& sb = built[(size_t)sw];
                const int32_t* trk = &st[(size_t)sw * NT];
                if (trk[0] >= 0) { sb.group = group[trk[0]]; sb.perp = perp[trk[0]]; }
                int64_t remaining = 0;
                for (int b = 0; b < NT; ++b) {
                    if (trk[b] >= 0) { cur[b] = off[trk[b]]; endk[b] = off[trk[b] + 1]; lam[b] = lam0[trk[b]]; ++sb.n_active; }
                    else { cur[b] = endk[b] = 0; lam[b] = 0.0; }
                    remaining += endk[b] - cur[b];
                }
                sb.n_seg = remaining;
                while (remaining > 0) {
                    if (++tile_serial == INT32_MAX) { std::fill(stamp.begin(), stamp.end(), -1); tile_serial = 0; }
                    regions.clear();
                    rcount.clear();
                    for (int b = 0; b < NT; ++b) { first[b] = cur[b]; cnt[b] = 0; }
                    int nseg = 0;
                    auto take = [&](int b) -> bool {   // next segment of track b into the tile; false: region window full
                        const int64_t k = cur[b];
                        const int32_t r = desc->seg_region[k];
                        if (stamp[r] != tile_serial) {
                            if ((int)regions.size() == Lmax) return false;
                            stamp[r] = tile_serial;
                            lidx[r] = (int32_t)regions.size();
                            regions.push_back((uint32_t)r);
                            rcount.push_back(0);
                        }
                        ++rcount[lidx[r]];
                        lam[b] += desc->seg_length[k];
                        ++cur[b]; ++cnt[b]; ++nseg; --remaining;
                        return true;
                    };
                    bool level = false;
                    if (lag_len >= 0.0) {
                        double lo = 0.0, hi = 0.0;
                        bool any = false;
                        for (int b = 0; b < NT; ++b)
                            if (cur[b] < endk[b]) {
                                if (!any) { lo = hi = lam[b]; any = true; }
                                else { lo = std::min(lo, lam[b]); hi = std::max(hi, lam[b]); }
                            }
                        level = hi - lo <= lag_len;
                    }
                    if (level) {   // equal counts: round j gives every unfinished track its j-th segment
                        bool full = false;
                        for (int j = 0; j < Kmax && !full && remaining > 0; ++j)
                            for (int b = 0; b < NT; ++b)
                                if (cur[b] < endk[b] && cnt[b] == j && !take(b)) { full = true; break; }
                    } else {       // geometric: the track furthest behind advances
                        for (;;) {
                            int bs = -1;
                            for (int b = 0; b < NT; ++b)
                                if (cur[b] < endk[b] && (bs < 0 || lam[b] < lam[bs])) bs = b;
                            if (bs < 0 || cnt[bs] == Kmax || !take(bs)) break;
                        }
                    }
                    // ---- encode ----
                    const int L = (int)regions.size();
                    {   // regions in descending order of their segment count: the flush units of one pass have lists of similar length
                        perm.resize(L);
                        std::iota(perm.begin(), perm.end(), 0);
                        std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return rcount[a] > rcount[b]; });
                        sorted_regions.resize(L); sorted_count.resize(L);
                        for (int l = 0; l < L; ++l) { sorted_regions[l] = regions[perm[l]]; sorted_count[l] = rcount[perm[l]]; lidx[regions[perm[l]]] = l; }
                        regions.swap(sorted_regions); rcount.swap(sorted_count);
                    }
                    const int o_ss = 16;
                    const int o_rg = o_ss + nd_swath_pad16(2 * (NT + 1));
                    const int o_rc = o_rg + nd_swath_pad16(8 * L);   // = head bytes
                    const int bytes = o_rc + 16 * nseg;
                    const size_t base = sb.bytes.size();
                    sb.chunk_rel.push_back((uint32_t)(base / 16));
                    sb.head16.push_back((uint32_t)(o_rc / 16));
                    sb.bytes.resize(base + (size_t)bytes, 0);
                    uint8_t* c = sb.bytes.data() + base;
                    const uint32_t hdr[4] = {(uint32_t)L | ((uint32_t)nseg << 16), (uint32_t)(o_rg / 16),
                                             (uint32_t)o_rc, (uint32_t)bytes};
                    memcpy(c, hdr, 16);
                    uint16_t* ss = reinterpret_cast<uint16_t*>(c + o_ss);
                    uint32_t* rg = reinterpret_cast<uint32_t*>(c + o_rg);
                    uint32_t* rc = reinterpret_cast<uint32_t*>(c + o_rc);
                    rfill.resize(L);
                    for (int l = 0, e = 0; l < L; ++l) {
                        rfill[l] = e;
                        rg[2 * l] = regions[l];
                        rg[2 * l + 1] = (uint32_t)e | ((uint32_t)(e + rcount[l]) << 16);
                        e += rcount[l];
                    }
                    int o = 0, max_cnt = 0;
                    for (int b = 0; b < NT; ++b) {
                        ss[b] = (uint16_t)o;
                        max_cnt = std::max(max_cnt, cnt[b]);
                        for (int j = 0; j < cnt[b]; ++j, ++o) {
                            const int64_t k = first[b] + j;
                            const int32_t r = desc->seg_region[k];
                            const int l = lidx[r];
                            const float len = (float)desc->seg_length[k];
                            uint32_t lenbits;
                            memcpy(&lenbits, &len, 4);
                            rc[4 * o] = lenbits;
                            rc[4 * o + 1] = (uint32_t)(l * line_q);
                            rc[4 * o + 2] = (uint32_t)(desc->region_material[r] * line);
                            rc[4 * o + 3] = (uint32_t)(rfill[l]++ * row_bytes);   // region-major delta row: by slot, then along the track
                        }
                    }
                    ss[NT] = (uint16_t)o;
                    if (prm.keep_slot_start) sb.slot_start.insert(sb.slot_start.end(), ss, ss + NT + 1);
                    sb.sum_regions += L;
                    sb.sum_max_cnt += max_cnt;
                    sb.max_head = std::max(sb.max_head, o_rc);
                    sb.max_rec = std::max(sb.max_rec, 16 * nseg);
                }
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
        if (byte0[n_sw] / 16 >= 0xffffffffull) return nd_fail(ND_ERR_RANGE, "swath stream exceeds 64 GiB");
        out->tile_ref.resize((size_t)out->n_tiles + 1);
        out->tile_ref[(size_t)out->n_tiles] = {(uint32_t)(byte0[n_sw] / 16), 0u};   // end sentinel: chunk k spans [k, k+1)
        out->blob.resize_uninitialised(byte0[n_sw]);   // first touched by the parallel copies below
        int64_t sum_regions = 0, sum_seg = 0, sum_slots = 0;
        int max_head = 0, max_rec = 0;
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            sum_regions += built[sw].sum_regions; sum_seg += built[sw].n_seg;
            max_head = std::max(max_head, built[sw].max_head); max_rec = std::max(max_rec, built[sw].max_rec);
            sum_slots += built[sw].sum_max_cnt * built[sw].n_active;
        }
#pragma omp parallel for schedule(dynamic, 64) num_threads(nth)
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            SwathBuild& sb = built[(size_t)sw];
            if (!sb.bytes.empty()) memcpy(out->blob.data() + byte0[sw], sb.bytes.data(), sb.bytes.size());
            const uint32_t b16 = (uint32_t)(byte0[sw] / 16);
            for (size_t i = 0; i < sb.chunk_rel.size(); ++i)
                out->tile_ref[(size_t)out->swath_tile0[sw] + i] = {b16 + sb.chunk_rel[i], sb.head16[i]};
            std::vector<uint8_t>().swap(sb.bytes);
        }
        if (prm.keep_slot_start) {
            out->slot_start.resize((size_t)out->n_tiles * (NT + 1));
#pragma omp parallel for schedule(dynamic, 64) num_threads(nth)
            for (int64_t sw = 0; sw < n_sw; ++sw) {
                SwathBuild& sb = built[(size_t)sw];
                if (!sb.slot_start.empty())
                    memcpy(out->slot_start.data() + (size_t)out->swath_tile0[sw] * (NT + 1), sb.slot_start.data(), sizeof(uint16_t) * sb.slot_start.size());
                std::vector<uint16_t>().swap(sb.slot_start);
            }
        }
        out->max_head_bytes = max_head;
        out->max_rec_bytes = max_rec;
        out->mean_regions_per_tile = out->n_tiles ? (double)sum_regions / (double)out->n_tiles : 0.0;
        out->mean_segments_per_tile = out->n_tiles ? (double)sum_seg / (double)out->n_tiles : 0.0;
        out->lockstep_efficiency = sum_slots ? (double)sum_seg / (double)sum_slots : 1.0;
        // ---- 5. work items (swath, direction) ----
        out->items.clear();
        if (prm.item_order == 0) {   // most expensive first
            for (int64_t sw = 0; sw < n_sw; ++sw) {
                const int32_t c32 = (int32_t)std::min<int64_t>(built[sw].sum_max_cnt, INT32_MAX);
                out->items.push_back({(int32_t)sw, 0, c32, 0});
                out->items.push_back({(int32_t)sw, 1, c32, 0});
            }
            std::stable_sort(out->items.begin(), out->items.end(), [](const NdSwathItem& a, const NdSwathItem& b) { return a.cost > b.cost; });
        } else {
            // Angle by angle; inside an angle all forward items in the order of the perpendicular coordinate, then all
            // backward items: thread blocks that run at the same time carry neighbouring swaths at the same stage of their
            // tracks, so the q and tally rows of the triangles two swaths share are still in L2 for the second one.  Swaths
            // are already stored in (angle, perpendicular) order; the last items of the last angle are short corner swaths.
            for (int64_t a = 0; a < n_sw;) {
                int64_t b = a;
                while (b < n_sw && built[b].group == built[a].group) ++b;
                for (int dir = 0; dir < 2; ++dir)
                    for (int64_t sw = a; sw < b; ++sw)
                        out->items.push_back({(int32_t)sw, dir, (int32_t)std::min<int64_t>(built[sw].sum_max_cnt, INT32_MAX), 0});
                a = b;
            }
        }
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_build_swaths: out of host memory");
    }
    return ND_OK;
}

// ------------------------------------------------------------------------------------------------
// C ABI access to the stream (include/nd.h "Diagnostics"): lets host-side tests decode every chunk.
// ------------------------------------------------------------------------------------------------
struct nd_swath_stream {
    NdSwathSet set;
};

extern "C" nd_status nd_swath_stream_build(const nd_problem_desc* desc, int32_t tracks_per_swath, int32_t tile_segments,
                                           int32_t window_regions, int32_t slots_per_line, int32_t row_bytes,
                                           double lag_segments, int32_t item_order, nd_swath_stream** out)
{
    if (!desc || !out) return nd_fail(ND_ERR_NULL, "nd_swath_stream_build: NULL argument");
    if (!desc->track_seg_offset || !desc->seg_region || !desc->seg_length || !desc->region_material)
        return nd_fail(ND_ERR_NULL, "nd_swath_stream_build: a descriptor array is NULL");
    if ((desc->track_azim == nullptr) != (desc->track_ends == nullptr))
        return nd_fail(ND_ERR_INVALID, "track_azim and track_ends must both be set or both be NULL");
    nd_swath_stream* s = new (std::nothrow) nd_swath_stream();
    if (!s) return nd_fail(ND_ERR_NOMEM, "nd_swath_stream_build: out of host memory");
    NdSwathParams prm{tracks_per_swath, tile_segments, window_regions, slots_per_line, row_bytes, lag_segments};
    prm.item_order = item_order;
    const nd_status rc = nd_build_swaths(desc, desc->track_azim, desc->track_ends, prm, 0, &s->set);
    if (rc != ND_OK) { delete s; return rc; }
    *out = s;
    return ND_OK;
}

extern "C" nd_status nd_swath_stream_view(const nd_swath_stream* s, nd_swath_stream_view_t* v)
{
    if (!s || !v) return nd_fail(ND_ERR_NULL, "nd_swath_stream_view: NULL argument");
    const NdSwathSet& t = s->set;
    v->n_swaths = t.n_swaths; v->n_tiles = t.n_tiles; v->blob_bytes = (int64_t)t.blob.size();
    v->n_items = (int64_t)t.items.size();
    static_assert(sizeof(NdSwathTileRef) == 8, "tile reference layout");
    v->blob = t.blob.data(); v->tile_ref = reinterpret_cast<const uint32_t*>(t.tile_ref.data()); v->swath_tile0 = t.swath_tile0.data();
    v->swath_track = t.swath_track.data(); v->items = reinterpret_cast<const int32_t*>(t.items.data());
    v->mean_regions_per_tile = t.mean_regions_per_tile; v->mean_segments_per_tile = t.mean_segments_per_tile;
    v->lockstep_efficiency = t.lockstep_efficiency; v->max_head_bytes = t.max_head_bytes; v->max_rec_bytes = t.max_rec_bytes;
    return ND_OK;
}

extern "C" nd_status nd_swath_stream_destroy(nd_swath_stream* s)
{
    delete s;
    return ND_OK;
}

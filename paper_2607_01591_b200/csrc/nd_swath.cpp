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
#include "nd_swath_core.h"

namespace {

struct SwathBuild {
    std::vector<uint8_t> bytes;        // this swath's chunks, concatenated
    std::vector<uint32_t> ref;         // per chunk: offset from the swath's first byte, head size (16-B units)
    std::vector<uint16_t> slot_start;  // [tiles][NT+1] when requested
    int64_t n_seg = 0, sum_regions = 0, sum_max_cnt = 0, n_active = 0;
    int max_head = 0, max_rec = 0;
};

} // namespace

// The length under which the fronts of a swath's tracks count as level: `lag` mean segment lengths.  With track geometry the
// mean is (sum of the tracks' end-to-end lengths) / S, formed in track order on the host -- the same number whether the
// segments live on the host or on the device; without geometry it is the mean of the segment lengths themselves.
double nd_swath_lag_length(const nd_problem_desc* desc, const double* track_ends, double lag, int n_threads)
{
    if (lag < 0.0) return -1.0;
    const int T = desc->n_tracks;
    const int64_t S = desc->track_seg_offset[T];
    if (S <= 0) return 0.0;
    double sum = 0.0;
    if (track_ends) {
        for (int t = 0; t < T; ++t) {
            if (desc->track_seg_offset[t + 1] == desc->track_seg_offset[t]) continue;
            const double dx = track_ends[4 * (size_t)t + 2] - track_ends[4 * (size_t)t], dy = track_ends[4 * (size_t)t + 3] - track_ends[4 * (size_t)t + 1];
            const double h = std::sqrt(dx * dx + dy * dy);
            if (std::isfinite(h)) sum += h;
        }
    } else {
#pragma omp parallel for reduction(+ : sum) num_threads(n_threads > 0 ? n_threads : 1)
        for (int64_t k = 0; k < S; ++k) sum += desc->seg_length[k];
    }
    return lag * sum / (double)S;
}

nd_status nd_swath_check_params(const nd_problem_desc* desc, const NdSwathParams& prm, NdSwathCoreParams* core)
{
    const int NT = prm.NT, Kmax = prm.Kmax, Lmax = prm.Lmax, NC = prm.NC;
    if (NT < 1 || NT > 1024 || Kmax < 1 || Lmax < 1 || NC < 1 || NT % NC != 0 || prm.row_bytes < 16 || prm.row_bytes % 16 != 0)
        return nd_fail(ND_ERR_INVALID, "swath parameters out of range");
    const int64_t line = (int64_t)NC * prm.row_bytes;   // bytes between consecutive sigma_t rows in shared memory
    const int NCq = prm.NCq > 0 ? prm.NCq : NC;
    const int64_t line_q = (int64_t)NCq * prm.row_bytes; // bytes between consecutive q rows
    if (Lmax > 65535 || (int64_t)NT * Kmax > 65535 || nd_swath_head_capacity(prm) / 16 > 65535 ||
        (int64_t)Lmax * line_q > (1ll << 30) || (int64_t)desc->n_materials * line > (1ll << 30))
        return nd_fail(ND_ERR_INVALID, "swath parameters: tile sizes must fit 16 bits");
    core->NT = NT; core->Kmax = Kmax; core->Lmax = Lmax; core->line = line; core->line_q = line_q;
    core->row_bytes = prm.row_bytes;   // bytes between consecutive delta rows
    core->lag_len = -1.0;
    return ND_OK;
}

// Steps 1 and 2 of the build, which need the track geometry but no segment: which tracks share a swath.
nd_status nd_swath_plan(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends, const NdSwathParams& prm,
                        NdSwathPlan* plan)
{
    const int T = desc->n_tracks, NT = prm.NT;
    try {
        // ---- 1. order tracks: by angle id, then by perpendicular coordinate ----
        std::vector<int32_t> order(T);
        std::iota(order.begin(), order.end(), 0);
        std::vector<double> perp(T, 0.0);
        std::vector<int32_t> group(T, 0);
        plan->lam0.assign((size_t)T, 0.0);
        std::vector<double>& lam0 = plan->lam0;
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
        std::vector<int32_t>& st = plan->swath_track;
        st.clear();
        plan->group.clear();
        for (int i = 0; i < T;) {
            int n = 0;
            const int g = group[order[i]];
            while (n < NT && i + n < T && group[order[i + n]] == g) ++n;
            for (int b = 0; b < NT; ++b) st.push_back(b < n ? order[i + b] : -1);
            plan->group.push_back(g);
            i += n;
        }
        plan->n_swaths = (int64_t)(st.size() / NT);
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_swath_plan: out of host memory");
    }
    return ND_OK;
}

// Step 5: the work items (swath, direction) from every swath's cost (sum over its tiles of the longest slot).
void nd_swath_items(const NdSwathPlan& plan, const int64_t* cost, int item_order, std::vector<NdSwathItem>* items)
{
    const int64_t n_sw = plan.n_swaths;
    items->clear();
    if (item_order == 0) {   // most expensive first
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            const int32_t c32 = (int32_t)std::min<int64_t>(cost[sw], INT32_MAX);
            items->push_back({(int32_t)sw, 0, c32, 0});
            items->push_back({(int32_t)sw, 1, c32, 0});
        }
        std::stable_sort(items->begin(), items->end(), [](const NdSwathItem& a, const NdSwathItem& b) { return a.cost > b.cost; });
    } else {
        // Angle by angle; inside an angle all forward items in the order of the perpendicular coordinate, then all
        // backward items: thread blocks that run at the same time carry neighbouring swaths at the same stage of their
        // tracks, so the q and tally rows of the triangles two swaths share are still in L2 for the second one.  Swaths
        // are already stored in (angle, perpendicular) order; the last items of the last angle are short corner swaths.
        for (int64_t a = 0; a < n_sw;) {
            int64_t b = a;
            while (b < n_sw && plan.group[(size_t)b] == plan.group[(size_t)a]) ++b;
            for (int dir = 0; dir < 2; ++dir)
                for (int64_t sw = a; sw < b; ++sw)
                    items->push_back({(int32_t)sw, dir, (int32_t)std::min<int64_t>(cost[sw], INT32_MAX), 0});
            a = b;
        }
    }
}

nd_status nd_build_swaths(const nd_problem_desc* desc, const int32_t* track_azim, const double* track_ends,
                          const NdSwathParams& prm, int n_threads, NdSwathSet* out)
{
    const int NT = prm.NT, Kmax = prm.Kmax, Lmax = prm.Lmax;
    NdSwathCoreParams cp{};
    nd_status rc0 = nd_swath_check_params(desc, prm, &cp);
    if (rc0 != ND_OK) return rc0;
    NdSwathPlan plan;
    rc0 = nd_swath_plan(desc, track_azim, track_ends, prm, &plan);
    if (rc0 != ND_OK) return rc0;
    try {
        out->prm = prm;
        out->swath_track = plan.swath_track;
        const std::vector<int32_t>& st = out->swath_track;
        const std::vector<double>& lam0 = plan.lam0;
        const int64_t n_sw = plan.n_swaths;
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
        const double lag_len = nd_swath_lag_length(desc, track_ends, prm.lag, nth);
        cp.lag_len = lag_len;
        const int head_cap = nd_swath_head_capacity(prm), min_tile = Kmax < Lmax ? Kmax : Lmax;
        bool oom = false;
#pragma omp parallel num_threads(nth)
        {
            // the cutter / encoder of one swath is nd_swath_core (shared with the device builder); it fills a thread-local
            // buffer sized for the swath's upper bound, the used part is kept
            std::vector<uint8_t> scratch((size_t)nd_swath_scratch_bytes(NT, Kmax, Lmax)), tmp;
            std::vector<uint32_t> ref;
            std::vector<uint16_t> sst;
            const NdSwathScratch sc = nd_swath_scratch_at(scratch.data(), NT, Kmax, Lmax);
#pragma omp for schedule(dynamic, 4)
            for (int64_t sw = 0; sw < n_sw; ++sw) {
                if (oom) continue;
                SwathBuild& sb = built[(size_t)sw];
                const int32_t* trk = &st[(size_t)sw * NT];
                int64_t n_seg = 0;
                for (int b = 0; b < NT; ++b)
                    if (trk[b] >= 0) n_seg += off[trk[b] + 1] - off[trk[b]];
                const int64_t max_tiles = n_seg / min_tile + NT + 1;
                const size_t bound = 16 * (size_t)n_seg + (size_t)max_tiles * head_cap;
                try {
                    if (tmp.size() < bound) tmp.resize(bound);
                    if ((int64_t)ref.size() < 2 * max_tiles) ref.resize(2 * (size_t)max_tiles);
                    if (prm.keep_slot_start && sst.size() < (size_t)max_tiles * (NT + 1)) sst.resize((size_t)max_tiles * (NT + 1));
                    memset(tmp.data(), 0, bound);
                    NdSwathCoreOut co{};
                    nd_swath_core<true>(cp, off, desc->seg_region, desc->seg_length, desc->region_material, trk, lam0.data(), sc, tmp.data(),
                                        ref.data(), 0u, prm.keep_slot_start ? sst.data() : nullptr, &co);
                    sb.bytes.assign(tmp.begin(), tmp.begin() + (size_t)co.n_bytes);
                    sb.ref.assign(ref.begin(), ref.begin() + 2 * (size_t)co.n_tiles);
                    if (prm.keep_slot_start) sb.slot_start.assign(sst.begin(), sst.begin() + (size_t)co.n_tiles * (NT + 1));
                    sb.n_seg = co.n_seg; sb.sum_regions = co.sum_regions; sb.sum_max_cnt = co.sum_max_cnt; sb.n_active = co.n_active;
                    sb.max_head = co.max_head; sb.max_rec = co.max_rec;
                } catch (const std::bad_alloc&) {
#pragma omp atomic write
                    oom = true;
                }
            }
        }
        if (oom) return nd_fail(ND_ERR_NOMEM, "nd_build_swaths: out of host memory");
        // ---- 4. concatenate ----
        out->swath_tile0.assign((size_t)n_sw + 1, 0);
        std::vector<size_t> byte0((size_t)n_sw + 1, 0);
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            out->swath_tile0[sw + 1] = out->swath_tile0[sw] + (int64_t)(built[sw].ref.size() / 2);
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
            for (size_t i = 0; i < sb.ref.size() / 2; ++i)
                out->tile_ref[(size_t)out->swath_tile0[sw] + i] = {b16 + sb.ref[2 * i], sb.ref[2 * i + 1]};
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
        std::vector<int64_t> cost((size_t)n_sw);
        for (int64_t sw = 0; sw < n_sw; ++sw) cost[(size_t)sw] = built[(size_t)sw].sum_max_cnt;
        nd_swath_items(plan, cost.data(), prm.item_order, &out->items);
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

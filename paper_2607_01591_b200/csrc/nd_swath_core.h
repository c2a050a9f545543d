// nd_swath_core.h -- the tile cutter and chunk encoder of ONE swath (row A1; format: nd_swath.h), written once for both
// builders of the stream: the host builder (nd_swath.cpp, g++, a thread per swath under OpenMP) and the device builder
// (nd_swath_device.cu, a CUDA thread per swath).  The two therefore produce the same bytes; the host one is the checker
// (tests/test_gpu_stream_device.py compares the blobs byte for byte).
//
// COUNT pass (FILL = false): number of tiles and bytes of the swath.  FILL pass: the chunks, their offsets, their head sizes
// and (optionally) the slot_start arrays.  All scratch is caller-provided (host: vectors, device: a slice of the workspace).
#ifndef ND_SWATH_CORE_H
#define ND_SWATH_CORE_H
#include <stdint.h>

#ifdef __CUDACC__
#define ND_HD __host__ __device__ __forceinline__
#else
#define ND_HD inline
#endif

struct NdSwathCoreParams {
    int NT, Kmax, Lmax;
    int64_t line;        // bytes between consecutive Sigma_t rows in shared memory
    int64_t line_q;      // bytes between consecutive staged q rows
    int64_t row_bytes;   // bytes between consecutive delta rows
    double lag_len;      // >= 0: equal-count tiles while the fronts lie within this length of each other; < 0: always geometric
};

struct NdSwathCoreOut {
    int64_t n_tiles, n_bytes, n_seg, sum_regions, sum_max_cnt;
    int32_t n_active, max_head, max_rec, reserved;
};

// scratch of one swath: int64 cur/first/endk [NT]; double lam [NT]; int32 cnt [NT], regions/rcount/order/newidx/rfill [Lmax];
// uint16 seg_l [NT * Kmax]
ND_HD int64_t nd_swath_scratch_bytes(int NT, int Kmax, int Lmax)
{
    const int64_t b = 8 * 3 * (int64_t)NT + 8 * (int64_t)NT + 4 * (int64_t)NT + 4 * 5 * (int64_t)Lmax + 2 * (int64_t)NT * Kmax;
    return (b + 15) / 16 * 16;
}

struct NdSwathScratch {
    int64_t *cur, *first, *endk;
    double* lam;
    int32_t *cnt, *regions, *rcount, *order, *newidx, *rfill;
    uint16_t* seg_l;
};

ND_HD NdSwathScratch nd_swath_scratch_at(void* base, int NT, int Kmax, int Lmax)
{
    NdSwathScratch s;
    char* p = static_cast<char*>(base);
    s.cur = reinterpret_cast<int64_t*>(p); p += 8 * (int64_t)NT;
    s.first = reinterpret_cast<int64_t*>(p); p += 8 * (int64_t)NT;
    s.endk = reinterpret_cast<int64_t*>(p); p += 8 * (int64_t)NT;
    s.lam = reinterpret_cast<double*>(p); p += 8 * (int64_t)NT;
    s.cnt = reinterpret_cast<int32_t*>(p); p += 4 * (int64_t)NT;
    s.regions = reinterpret_cast<int32_t*>(p); p += 4 * (int64_t)Lmax;
    s.rcount = reinterpret_cast<int32_t*>(p); p += 4 * (int64_t)Lmax;
    s.order = reinterpret_cast<int32_t*>(p); p += 4 * (int64_t)Lmax;
    s.newidx = reinterpret_cast<int32_t*>(p); p += 4 * (int64_t)Lmax;
    s.rfill = reinterpret_cast<int32_t*>(p); p += 4 * (int64_t)Lmax;
    s.seg_l = reinterpret_cast<uint16_t*>(p);
    (void)Kmax;
    return s;
}

ND_HD int nd_swath_pad16_core(int x) { return (x + 15) / 16 * 16; }

// trk [NT]: track ids of the swath's slots (-1: empty slot); lam0 [T]: coordinate of every track's start point along the
// direction of its angle.  FILL: `bytes` points at the swath's first chunk (16-byte aligned, zero-filled by the caller),
// tile_ref [n_tiles][2] receives every chunk's { base16 + offset from there, head size } in 16-byte units, slot_start_out
// (may be NULL) [n_tiles][NT+1].
template <bool FILL>
ND_HD void nd_swath_core(const NdSwathCoreParams& P, const int64_t* off, const int32_t* seg_region, const double* seg_length,
                         const int32_t* region_material, const int32_t* trk, const double* lam0, const NdSwathScratch& s, uint8_t* bytes,
                         uint32_t* tile_ref, uint32_t base16, uint16_t* slot_start_out, NdSwathCoreOut* out)
{
    const int NT = P.NT, Kmax = P.Kmax, Lmax = P.Lmax;
    NdSwathCoreOut o;
    o.n_tiles = 0; o.n_bytes = 0; o.n_seg = 0; o.sum_regions = 0; o.sum_max_cnt = 0; o.n_active = 0; o.max_head = 0; o.max_rec = 0; o.reserved = 0;
    int64_t remaining = 0;
    for (int b = 0; b < NT; ++b) {
        if (trk[b] >= 0) { s.cur[b] = off[trk[b]]; s.endk[b] = off[trk[b] + 1]; s.lam[b] = lam0[trk[b]]; ++o.n_active; }
        else { s.cur[b] = 0; s.endk[b] = 0; s.lam[b] = 0.0; }
        remaining += s.endk[b] - s.cur[b];
    }
    o.n_seg = remaining;
    while (remaining > 0) {
        int L = 0, nseg = 0;
        for (int b = 0; b < NT; ++b) { s.first[b] = s.cur[b]; s.cnt[b] = 0; }
        // next segment of track b into the tile; false: the region window is full
        auto take = [&](int b) -> bool {
            const int64_t k = s.cur[b];
            const int32_t r = seg_region[k];
            int l = L - 1;   // newest first: a track stays in a region for a few segments and its neighbours follow it
            while (l >= 0 && s.regions[l] != r) --l;
            if (l < 0) {
                if (L == Lmax) return false;
                l = L;
                s.regions[L] = r; s.rcount[L] = 0; ++L;
            }
            ++s.rcount[l];
            s.seg_l[b * Kmax + s.cnt[b]] = (uint16_t)l;
            s.lam[b] += seg_length[k];
            ++s.cur[b]; ++s.cnt[b]; ++nseg; --remaining;
            return true;
        };
        bool level = false;
        if (P.lag_len >= 0.0) {
            double lo = 0.0, hi = 0.0;
            bool any = false;
            for (int b = 0; b < NT; ++b)
                if (s.cur[b] < s.endk[b]) {
                    if (!any) { lo = hi = s.lam[b]; any = true; }
                    else { lo = s.lam[b] < lo ? s.lam[b] : lo; hi = s.lam[b] > hi ? s.lam[b] : hi; }
                }
            level = hi - lo <= P.lag_len;
        }
        if (level) {   // equal counts: round j gives every unfinished track its j-th segment
            bool full = false;
            for (int j = 0; j < Kmax && !full && remaining > 0; ++j)
                for (int b = 0; b < NT; ++b)
                    if (s.cur[b] < s.endk[b] && s.cnt[b] == j && !take(b)) { full = true; break; }
        } else {       // geometric: the track furthest behind advances
            for (;;) {
                int bs = -1;
                for (int b = 0; b < NT; ++b)
                    if (s.cur[b] < s.endk[b] && (bs < 0 || s.lam[b] < s.lam[bs])) bs = b;
                if (bs < 0 || s.cnt[bs] == Kmax || !take(bs)) break;
            }
        }
        // ---- sizes ----
        const int o_ss = 16;
        const int o_rg = o_ss + nd_swath_pad16_core(2 * (NT + 1));
        const int o_rc = o_rg + nd_swath_pad16_core(8 * L);   // = head bytes
        const int nbytes = o_rc + 16 * nseg;
        int max_cnt = 0;
        for (int b = 0; b < NT; ++b) max_cnt = s.cnt[b] > max_cnt ? s.cnt[b] : max_cnt;
        if (FILL) {
            // regions in descending order of their segment count (stable insertion sort): the flush units of one pass have
            // lists of similar length
            for (int l = 0; l < L; ++l) {
                int i = l;
                while (i > 0 && s.rcount[s.order[i - 1]] < s.rcount[l]) { s.order[i] = s.order[i - 1]; --i; }
                s.order[i] = l;
            }
            for (int l = 0; l < L; ++l) s.newidx[s.order[l]] = l;
            uint8_t* c = bytes + o.n_bytes;
            uint32_t* hdr = reinterpret_cast<uint32_t*>(c);
            hdr[0] = (uint32_t)L | ((uint32_t)nseg << 16); hdr[1] = (uint32_t)(o_rg / 16); hdr[2] = (uint32_t)o_rc; hdr[3] = (uint32_t)nbytes;
            uint16_t* ss = reinterpret_cast<uint16_t*>(c + o_ss);
            uint32_t* rg = reinterpret_cast<uint32_t*>(c + o_rg);
            uint32_t* rc = reinterpret_cast<uint32_t*>(c + o_rc);
            for (int l = 0, e = 0; l < L; ++l) {
                const int old = s.order[l];
                s.rfill[l] = e;
                rg[2 * l] = (uint32_t)s.regions[old];
                rg[2 * l + 1] = (uint32_t)e | ((uint32_t)(e + s.rcount[old]) << 16);
                e += s.rcount[old];
            }
            int at = 0;
            for (int b = 0; b < NT; ++b) {
                ss[b] = (uint16_t)at;
                for (int j = 0; j < s.cnt[b]; ++j, ++at) {
                    const int64_t k = s.first[b] + j;
                    const int32_t r = seg_region[k];
                    const int l = s.newidx[s.seg_l[b * Kmax + j]];
                    const float len = (float)seg_length[k];
                    union { float f; uint32_t u; } cv;
                    cv.f = len;
                    rc[4 * at] = cv.u;
                    rc[4 * at + 1] = (uint32_t)(l * P.line_q);
                    rc[4 * at + 2] = (uint32_t)(region_material[r] * P.line);
                    rc[4 * at + 3] = (uint32_t)(s.rfill[l]++ * P.row_bytes);   // region-major delta row: by slot, then along the track
                }
            }
            ss[NT] = (uint16_t)at;
            tile_ref[2 * o.n_tiles] = base16 + (uint32_t)(o.n_bytes / 16);
            tile_ref[2 * o.n_tiles + 1] = (uint32_t)(o_rc / 16);
            if (slot_start_out)
                for (int b = 0; b <= NT; ++b) slot_start_out[o.n_tiles * (NT + 1) + b] = ss[b];
        }
        o.n_bytes += nbytes;
        ++o.n_tiles;
        o.sum_regions += L;
        o.sum_max_cnt += max_cnt;
        o.max_head = o_rc > o.max_head ? o_rc : o.max_head;
        o.max_rec = 16 * nseg > o.max_rec ? 16 * nseg : o.max_rec;
    }
    *out = o;
}

#endif

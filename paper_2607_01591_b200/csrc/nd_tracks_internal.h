// nd_tracks_internal.h -- private: the nd_tracks object and the host steps shared by nd_tracks_generate (host ray
// walk) and nd_tracks_generate_device (CUDA ray walk).  All FP64 geometry on the host lives in nd_tracks.cpp, which is
// compiled with -ffp-contract=off (rule R-T / R-W: bit-exact expression trees).
#ifndef ND_TRACKS_INTERNAL_H
#define ND_TRACKS_INTERNAL_H
#include <cstdint>
#include <memory>
#include <vector>

#include "nd.h"

// Array that is NOT value-initialised: the segment arrays of a 5e8-segment problem (5.8 GB) are written exactly once, by
// the parallel host walk or by device-to-host copies; std::vector::resize would zero-fill them first on one thread (~2 s).
template <class T>
struct NdRawArray {
    std::unique_ptr<T[]> p;
    size_t n = 0;
    void resize(size_t count) { p.reset(count ? new T[count] : nullptr); n = count; }
    T* data() { return p.get(); }
    const T* data() const { return p.get(); }
    size_t size() const { return n; }
    T& operator[](size_t i) { return p[i]; }
    const T& operator[](size_t i) const { return p[i]; }
};

// writes one byte per 4 KB page with all host threads: first touch of a freshly allocated array before a
// device-to-host copy fills it (the copy would otherwise fault the pages in one by one)
void nd_touch_pages(void* p, size_t bytes);

struct NdAngleSet {          // one track angle j in (0, pi)
    int nx = 0, ny = 0;      // tracks leaving the bottom side / the vertical side
    double dx = 0, dy = 0;   // slot widths
    double ux = 0, uy = 0;   // unit forward direction (uy > 0)
    double delta = 0;        // effective spacing
    double phi = 0;          // effective angle of the first-quadrant partner
    double omega = 0;        // azimuthal weight per direction
    int first = 0;           // id of the angle's first track
    bool mirrored = false;   // second quadrant (ux < 0)
};

struct nd_tracks {
    int n_azim = 0, n_half = 0, n_tracks = 0, n_regions = 0;
    int64_t n_segments = 0;
    std::vector<NdAngleSet> angles;
    std::vector<int64_t> seg_offset;
    NdRawArray<int32_t> seg_region;   // every element written by the walk
    NdRawArray<double> seg_length;
    std::vector<double> track_weight;
    std::vector<int32_t> link;
    std::vector<int32_t> track_azim;
    std::vector<double> ends;
    std::vector<double> volume;
    std::vector<double> azim_phi, azim_weight, azim_spacing;
    std::vector<int32_t> global_id;   // [T] id of every track in the unsharded laydown (identity unless made by nd_tracks_shard)
    // nd_tracks_generate_resident: the segment arrays in the caller's device workspace; the host arrays above stay empty
    // until nd_tracks_materialise
    const int32_t* d_seg_region = nullptr;
    const double* d_seg_length = nullptr;
    bool host_segments = true;
};

// What a ray walker needs besides the mesh arrays: the half-edge twins and every track's first triangle.
struct NdWalkInput {
    std::vector<int32_t> twin;        // [3R] opposite half-edge or -1
    std::vector<int32_t> start_tri;   // [T]  triangle that holds the track's start point (rule R-W)
};

// Laydown (R-T), links (O-3), half-edge mesh and start triangles.  *out owns the result (segments still empty).
nd_status nd_tracks_prepare(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, nd_tracks** out, NdWalkInput* walk);
// After seg_offset / seg_region / seg_length are filled: track volumes (O-5, canonical order; skipped with
// volumes_from_segments = false: the caller fills tr->volume) and the per-angle views.
nd_status nd_tracks_finish(nd_tracks* tr, bool volumes_from_segments = true);

#endif

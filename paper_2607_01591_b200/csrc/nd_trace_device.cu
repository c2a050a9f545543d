// nd_trace_device.cu -- SURVEY.md section 8(f) NEXT-1: the ray-mesh intersection (rule R-W) on the GPU.
//
// Laydown, links, the half-edge twins and every track's first triangle come from the host code in nd_tracks.cpp
// (nd_tracks_prepare: integer rules + a few FP64 operations per angle); the WALK -- by far the largest part, one step per
// segment -- runs here, one thread per track, in two passes (count, then fill) like the host walker.  The FP64
// expression trees are the ones rule R-W fixes, written with the round-to-nearest intrinsics (__dmul_rn, __dsub_rn,
// __ddiv_rn), which the compiler never contracts into FMAs: the result is bit-identical to the host walker's and to
// the oracle's (tests memcmp all three).
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "nd.h"
#include "nd_internal.h"
#include "nd_tracks_internal.h"

namespace {

struct WalkParams {
    const double* __restrict__ xy;         // [V][2]
    const int32_t* __restrict__ tri;       // [R][3]
    const int32_t* __restrict__ twin;      // [3R]
    const double* __restrict__ trk;        // [T][4] x0, y0, ux, uy
    const int32_t* __restrict__ start_tri; // [T]
    const int64_t* __restrict__ seg_off;   // [T+1] (fill pass)
    int64_t* __restrict__ counts;          // [T]   (count pass; -1 = the walk left the mesh)
    int32_t* __restrict__ seg_region;      // fill pass: batch-local outputs
    double* __restrict__ seg_length;
    const double* __restrict__ w2;         // [T] 2 * track weight   } resident fill pass: A~_r += 2 omega_a delta_a s (O-5)
    double* vol;                           // [R] or NULL            }
    int64_t guard, base;                   // max steps; seg_off of the batch's first track
    int t0, t1;
};

template <bool kStore>
__global__ void __launch_bounds__(128) k_walk(const WalkParams p)
{
    const int t = p.t0 + blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= p.t1) return;
    const double x0 = p.trk[4 * (size_t)t], y0 = p.trk[4 * (size_t)t + 1], ux = p.trk[4 * (size_t)t + 2], uy = p.trk[4 * (size_t)t + 3];
    int tr = p.start_tri[t];
    double lam_prev = 0.0;
    int64_t count = 0;
    int32_t* reg = nullptr;
    double* len = nullptr;
    double w2 = 0.0;
    if (kStore) {
        reg = p.seg_region + (p.seg_off[t] - p.base); len = p.seg_length + (p.seg_off[t] - p.base);
        if (p.vol) w2 = p.w2[t];
    }
    bool ok = false;
    for (int64_t step = 0; step <= p.guard; ++step) {
        const int v[3] = {p.tri[3 * (size_t)tr], p.tri[3 * (size_t)tr + 1], p.tri[3 * (size_t)tr + 2]};
        double px[3], py[3];
#pragma unroll
        for (int e = 0; e < 3; ++e) { px[e] = p.xy[2 * (size_t)v[e]]; py[e] = p.xy[2 * (size_t)v[e] + 1]; }
        int exit_e = -1;
        double lam_exit = 0.0;
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int f = (e + 1) % 3;
            const double ex = __dsub_rn(px[f], px[e]), ey = __dsub_rn(py[f], py[e]);          // CCW edge of the triangle
            const double facing = __dsub_rn(__dmul_rn(ux, ey), __dmul_rn(uy, ex));           // u . outward normal
            if (!(facing > 0.0)) continue;
            const bool fwd = v[e] < v[f];                                                      // canonical orientation: lower id first
            const double ax = fwd ? px[e] : px[f], ay = fwd ? py[e] : py[f];
            const double bx = fwd ? px[f] : px[e], by = fwd ? py[f] : py[e];
            const double Ex = __dsub_rn(bx, ax), Ey = __dsub_rn(by, ay);
            const double den = __dsub_rn(__dmul_rn(ux, Ey), __dmul_rn(uy, Ex));
            const double num = __dsub_rn(__dmul_rn(__dsub_rn(ax, x0), Ey), __dmul_rn(__dsub_rn(ay, y0), Ex));
            const double lam = __ddiv_rn(num, den);
            if (exit_e < 0 || lam < lam_exit) { exit_e = e; lam_exit = lam; }                  // ties keep the lower edge
        }
        if (exit_e < 0) break;
        const double chord = __dsub_rn(lam_exit, lam_prev);
        if (chord > 0.0) {
            if (kStore) {
                reg[count] = tr; len[count] = chord;
                if (p.vol) atomicAdd(p.vol + tr, w2 * chord);
            }
            ++count;
        }
        lam_prev = lam_exit;
        const int32_t tw = p.twin[3 * (size_t)tr + exit_e];
        if (tw < 0) { ok = true; break; }
        tr = tw / 3;
    }
    if (!kStore) p.counts[t] = ok ? count : -1;
}

inline size_t up256(size_t x) { return (x + 255) / 256 * 256; }

struct TraceLayout { size_t xy, tri, twin, trk, start_tri, counts, seg_off, w2, vol, out, total_fixed; };

TraceLayout trace_layout(size_t V, size_t R, size_t T)
{
    TraceLayout L{};
    size_t c = 0;
    auto bump = [&](size_t bytes) { const size_t at = c; c = up256(c + bytes); return at; };
    L.xy = bump(16 * V); L.tri = bump(12 * R); L.twin = bump(12 * R); L.trk = bump(32 * T); L.start_tri = bump(4 * T);
    L.counts = bump(8 * T); L.seg_off = bump(8 * (T + 1)); L.w2 = bump(8 * T); L.vol = bump(8 * R);
    L.out = c; L.total_fixed = c;
    return L;
}

constexpr size_t kBytesPerSegment = 12;           // int32 region + double length
constexpr size_t kMinSegmentCapacity = 1u << 20;  // the longest single track must fit

} // namespace

#define ND_TRACE_CUDA(call)                                                                              \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            char buf_[512];                                                                              \
            snprintf(buf_, sizeof buf_, "%s failed: %s", #call, cudaGetErrorString(e_));                 \
            delete tr;                                                                                   \
            return nd_fail(ND_ERR_CUDA, buf_);                                                           \
        }                                                                                                \
    } while (0)

extern "C" nd_status nd_tracks_device_workspace_bytes(const nd_mesh_desc* mesh, int32_t n_azim, double spacing,
                                                      size_t* min_bytes, size_t* bytes_per_segment)
{
    if (!mesh || !min_bytes || !bytes_per_segment) return nd_fail(ND_ERR_NULL, "nd_tracks_device_workspace_bytes: NULL argument");
    if (mesh->n_vertices < 3 || mesh->n_triangles < 1 || !(mesh->W > 0.0) || !(mesh->H > 0.0) || !(spacing > 0.0) || n_azim < 4 ||
        n_azim % 4 != 0)
        return nd_fail(ND_ERR_INVALID, "nd_tracks_device_workspace_bytes: need V>=3, R>=1, W,H,spacing>0, n_azim a positive multiple of 4");
    // every angle has n_x + n_y tracks with n_x <= W/spacing + 1, n_y <= H/spacing + 1 (rule R-T)
    const double t_bound = 0.5 * n_azim * ((mesh->W + mesh->H) / spacing + 2.0);
    if (!(t_bound < 1.0e9)) return nd_fail(ND_ERR_RANGE, "nd_tracks_device_workspace_bytes: more than 1e9 tracks");
    const TraceLayout L = trace_layout((size_t)mesh->n_vertices, (size_t)mesh->n_triangles, (size_t)t_bound + 1);
    *min_bytes = L.total_fixed + kBytesPerSegment * kMinSegmentCapacity + 512;
    *bytes_per_segment = kBytesPerSegment;
    return ND_OK;
}

namespace {

nd_status trace_impl(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, void* device_workspace, size_t device_bytes,
                     void* cuda_stream, nd_trace_timing* timing, bool resident, size_t* required_bytes, nd_tracks** out)
{
    using clk = std::chrono::steady_clock;
    auto secs = [](clk::time_point a, clk::time_point b) { return std::chrono::duration<double>(b - a).count(); };
    const clk::time_point t_begin = clk::now();
    nd_trace_timing tm{};
    if (!out || !device_workspace) return nd_fail(ND_ERR_NULL, "nd_tracks_generate_device: NULL argument");
    if (reinterpret_cast<uintptr_t>(device_workspace) % 256 != 0) return nd_fail(ND_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    nd_tracks* tr = nullptr;
    NdWalkInput wi;
    nd_status rc = nd_tracks_prepare(mesh, n_azim, spacing, &tr, &wi);
    if (rc != ND_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    tm.prepare_s = secs(t_begin, clk::now());
    cudaEvent_t ev[2] = {nullptr, nullptr};
    try {
        ND_TRACE_CUDA(cudaEventCreate(&ev[0]));
        ND_TRACE_CUDA(cudaEventCreate(&ev[1]));
        const size_t V = (size_t)mesh->n_vertices, R = (size_t)mesh->n_triangles, T = (size_t)tr->n_tracks;
        const TraceLayout L = trace_layout(V, R, T);
        if (device_bytes < L.total_fixed + kBytesPerSegment * 1024) { delete tr; return nd_fail(ND_ERR_WORKSPACE, "workspace smaller than nd_tracks_device_workspace_bytes"); }
        // the output area holds `cap` segments: int32 regions first, then doubles (8-byte aligned)
        size_t cap = ((device_bytes - L.total_fixed) / kBytesPerSegment) & ~(size_t)63;
        char* ws = static_cast<char*>(device_workspace);
        std::vector<double> h_trk(4 * T);
        for (size_t t = 0; t < T; ++t) {
            const NdAngleSet& A = tr->angles[tr->track_azim[t]];
            h_trk[4 * t] = tr->ends[4 * t]; h_trk[4 * t + 1] = tr->ends[4 * t + 1]; h_trk[4 * t + 2] = A.ux; h_trk[4 * t + 3] = A.uy;
        }
        ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.xy, mesh->xy, 16 * V, cudaMemcpyHostToDevice, st));
        ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.tri, mesh->tri, 12 * R, cudaMemcpyHostToDevice, st));
        ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.twin, wi.twin.data(), 12 * R, cudaMemcpyHostToDevice, st));
        ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.trk, h_trk.data(), 32 * T, cudaMemcpyHostToDevice, st));
        ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.start_tri, wi.start_tri.data(), 4 * T, cudaMemcpyHostToDevice, st));
        WalkParams wp{};
        wp.xy = (const double*)(ws + L.xy); wp.tri = (const int32_t*)(ws + L.tri); wp.twin = (const int32_t*)(ws + L.twin);
        wp.trk = (const double*)(ws + L.trk); wp.start_tri = (const int32_t*)(ws + L.start_tri);
        wp.seg_off = (const int64_t*)(ws + L.seg_off); wp.counts = (int64_t*)(ws + L.counts);
        wp.seg_region = (int32_t*)(ws + L.out); wp.seg_length = (double*)(ws + L.out + 4 * cap);
        wp.guard = 4 * (int64_t)R + 16;
        // ---- pass 1: segment counts ----
        wp.t0 = 0; wp.t1 = (int)T;
        ND_TRACE_CUDA(cudaEventRecord(ev[0], st));
        k_walk<false><<<(unsigned)((T + 127) / 128), 128, 0, st>>>(wp);
        ND_TRACE_CUDA(cudaGetLastError());
        ND_TRACE_CUDA(cudaEventRecord(ev[1], st));
        std::vector<int64_t> h_counts(T);
        ND_TRACE_CUDA(cudaMemcpyAsync(h_counts.data(), wp.counts, 8 * T, cudaMemcpyDeviceToHost, st));
        ND_TRACE_CUDA(cudaStreamSynchronize(st));
        {
            float ms = 0.f;
            ND_TRACE_CUDA(cudaEventElapsedTime(&ms, ev[0], ev[1]));
            tm.count_kernel_ms = ms;
        }
        tr->seg_offset.assign(T + 1, 0);
        for (size_t t = 0; t < T; ++t) {
            if (h_counts[t] < 0) { delete tr; return nd_fail(ND_ERR_MESH, "nd_tracks_generate_device: ray walk left the mesh"); }
            tr->seg_offset[t + 1] = tr->seg_offset[t] + h_counts[t];
        }
        tr->n_segments = tr->seg_offset[T];
        ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.seg_off, tr->seg_offset.data(), 8 * (T + 1), cudaMemcpyHostToDevice, st));
        if (resident) {
            // all S segments stay in the workspace: regions, then lengths; A~_r is summed by the fill pass
            const size_t S = (size_t)tr->n_segments, need = L.total_fixed + up256(4 * S) + 8 * S + 512;
            if (required_bytes) *required_bytes = need;
            if (device_bytes < need) {
                char buf[160];
                snprintf(buf, sizeof buf, "nd_tracks_generate_resident: %lld segments need a workspace of %zu bytes", (long long)S, need);
                delete tr;
                cudaEventDestroy(ev[0]); cudaEventDestroy(ev[1]);
                return nd_fail(ND_ERR_WORKSPACE, buf);
            }
            std::vector<double> h_w2(T);
            for (size_t t = 0; t < T; ++t) h_w2[t] = 2.0 * tr->track_weight[t];
            ND_TRACE_CUDA(cudaMemcpyAsync(ws + L.w2, h_w2.data(), 8 * T, cudaMemcpyHostToDevice, st));
            ND_TRACE_CUDA(cudaMemsetAsync(ws + L.vol, 0, 8 * R, st));
            wp.w2 = (const double*)(ws + L.w2); wp.vol = (double*)(ws + L.vol);
            wp.seg_region = (int32_t*)(ws + L.out); wp.seg_length = (double*)(ws + L.out + up256(4 * S));
            wp.t0 = 0; wp.t1 = (int)T; wp.base = 0;
            ND_TRACE_CUDA(cudaEventRecord(ev[0], st));
            k_walk<true><<<(unsigned)((T + 127) / 128), 128, 0, st>>>(wp);
            ND_TRACE_CUDA(cudaGetLastError());
            ND_TRACE_CUDA(cudaEventRecord(ev[1], st));
            tr->volume.assign(R, 0.0);
            ND_TRACE_CUDA(cudaMemcpyAsync(tr->volume.data(), wp.vol, 8 * R, cudaMemcpyDeviceToHost, st));
            ND_TRACE_CUDA(cudaStreamSynchronize(st));
            float ms = 0.f;
            ND_TRACE_CUDA(cudaEventElapsedTime(&ms, ev[0], ev[1]));
            tm.fill_kernel_ms = ms;
            tm.batches = 1;
            tr->d_seg_region = wp.seg_region; tr->d_seg_length = wp.seg_length; tr->host_segments = false;
            cap = 0;
        } else {
            tr->seg_region.resize((size_t)tr->n_segments);
            tr->seg_length.resize((size_t)tr->n_segments);
            nd_touch_pages(tr->seg_region.data(), 4 * (size_t)tr->n_segments);
            nd_touch_pages(tr->seg_length.data(), 8 * (size_t)tr->n_segments);
        }
        // ---- pass 2: fill, in batches of tracks whose segments fit the output area ----
        for (size_t t0 = 0; t0 < T && !resident;) {
            size_t t1 = t0;
            while (t1 < T && (size_t)(tr->seg_offset[t1 + 1] - tr->seg_offset[t0]) <= cap) ++t1;
            if (t1 == t0) { delete tr; return nd_fail(ND_ERR_WORKSPACE, "nd_tracks_generate_device: one track has more segments than the workspace holds"); }
            const size_t n = (size_t)(tr->seg_offset[t1] - tr->seg_offset[t0]);
            wp.t0 = (int)t0; wp.t1 = (int)t1; wp.base = tr->seg_offset[t0];
            ND_TRACE_CUDA(cudaEventRecord(ev[0], st));
            k_walk<true><<<(unsigned)((t1 - t0 + 127) / 128), 128, 0, st>>>(wp);
            ND_TRACE_CUDA(cudaGetLastError());
            ND_TRACE_CUDA(cudaEventRecord(ev[1], st));
            const clk::time_point t_copy = clk::now();
            if (n > 0) {
                ND_TRACE_CUDA(cudaMemcpyAsync(tr->seg_region.data() + tr->seg_offset[t0], wp.seg_region, 4 * n, cudaMemcpyDeviceToHost, st));
                ND_TRACE_CUDA(cudaMemcpyAsync(tr->seg_length.data() + tr->seg_offset[t0], wp.seg_length, 8 * n, cudaMemcpyDeviceToHost, st));
            }
            ND_TRACE_CUDA(cudaStreamSynchronize(st));
            {
                float ms = 0.f;
                ND_TRACE_CUDA(cudaEventElapsedTime(&ms, ev[0], ev[1]));
                tm.fill_kernel_ms += ms;
                tm.copy_s += secs(t_copy, clk::now()) - 1e-3 * ms;
                ++tm.batches;
            }
            t0 = t1;
        }
        cudaEventDestroy(ev[0]);
        cudaEventDestroy(ev[1]);
    } catch (const std::bad_alloc&) {
        delete tr;
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_generate_device: out of host memory");
    }
    const clk::time_point t_fin = clk::now();
    rc = nd_tracks_finish(tr, !resident);
    if (rc != ND_OK) { delete tr; return rc; }
    tm.finish_s = secs(t_fin, clk::now());
    tm.total_s = secs(t_begin, clk::now());
    tm.n_segments = tr->n_segments;
    if (timing) *timing = tm;
    *out = tr;
    return ND_OK;
}

} // namespace

extern "C" nd_status nd_tracks_generate_device(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, void* device_workspace,
                                               size_t device_bytes, void* cuda_stream, nd_trace_timing* timing, nd_tracks** out)
{
    return trace_impl(mesh, n_azim, spacing, device_workspace, device_bytes, cuda_stream, timing, false, nullptr, out);
}

extern "C" nd_status nd_tracks_generate_resident(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, void* device_workspace,
                                                 size_t device_bytes, void* cuda_stream, nd_trace_timing* timing,
                                                 size_t* required_bytes, nd_tracks** out)
{
    return trace_impl(mesh, n_azim, spacing, device_workspace, device_bytes, cuda_stream, timing, true, required_bytes, out);
}

extern "C" nd_status nd_tracks_materialise(nd_tracks* tr, void* cuda_stream)
{
    if (!tr) return nd_fail(ND_ERR_NULL, "nd_tracks_materialise: NULL argument");
    if (tr->host_segments) return ND_OK;
    if (!tr->d_seg_region || !tr->d_seg_length) return nd_fail(ND_ERR_STATE, "nd_tracks_materialise: no device-resident segments");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const size_t S = (size_t)tr->n_segments;
    try {
        tr->seg_region.resize(S);
        tr->seg_length.resize(S);
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_materialise: out of host memory");
    }
    nd_touch_pages(tr->seg_region.data(), 4 * S);
    nd_touch_pages(tr->seg_length.data(), 8 * S);
    cudaError_t e = cudaSuccess;
    if (S > 0) {
        e = cudaMemcpyAsync(tr->seg_region.data(), tr->d_seg_region, 4 * S, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(tr->seg_length.data(), tr->d_seg_length, 8 * S, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        tr->seg_region.resize(0); tr->seg_length.resize(0);
        return nd_fail(ND_ERR_CUDA, cudaGetErrorString(e));
    }
    tr->host_segments = true;
    return ND_OK;
}

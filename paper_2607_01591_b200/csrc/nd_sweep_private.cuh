// nd_sweep_private.cuh -- row A2, the fast path: Eq. (5) with shared-memory private tallies.
//
// Why: on B200 one FP64 global RED per (segment, direction, group) runs at 3.5-5.9e11 /s while the arithmetic of
// the three polar updates behind it runs at 4.3e12/3 = 1.4e12 /s: global atomics per segment
// bind 2.4-4x before the exp pipe does.  Adjacent parallel tracks (0.01-0.05 cm apart) cross the same ~0.1-0.3 cm
// triangles, so a batch of B adjacent tracks re-visits every region ~B*delta/(B*delta+w) * w/delta times.
//
// Mapping
//   * lane group ("slot") = LPT = Gs/GPL lanes = one track at a time; each lane owns GPL consecutive groups and P polar
//     chains for each: GPL*P independent Eq.-(5) chains per lane (12 for GPL=4, P=3) -> ILP hides MUFU/FMA latency.
//   * a warp holds TPW = 32/LPT slots; slot s works on swath first_swath+s (B adjacent tracks of one angle), tile by
//     tile; a tile is one chunk (nd_tiles.h): <= Lw distinct regions, <= Nmax segments.
//   * per slot, in shared memory: the tile's chunk (double-buffered, staged by async copies one tile ahead), the q
//     rows of its L regions (async copies, 16-byte rows), and a PRIVATE FP32 tally window acc[L][Gs].  No other slot
//     ever touches it, so the accumulate is a plain LDS/FFMA/STS; the window is flushed with FP64 REDs once per tile.
//   * psi of the B tracks is carried between tiles in the psi_out array itself (L2-resident, 16-byte accesses,
//     prefetched one track ahead).
//   * persistent CTAs (one per SM), work items (TPW swaths x one direction) fetched from an atomic counter, most
//     expensive first.
#pragma once
#include "nd_kernels.cuh"

namespace ndk {

struct PrivParams {
    const uint8_t* __restrict__ blob;
    const uint32_t* __restrict__ tile_chunk;   // [n_tiles+1] chunk offsets in 16-byte units (+ end sentinel)
    const int64_t* __restrict__ swath_tile0;
    const int32_t* __restrict__ swath_track;
    const int4* __restrict__ items;
    int* __restrict__ counter;
    const float* __restrict__ q;
    const float* __restrict__ sigt;
    double* __restrict__ tally;
    const float* __restrict__ trk_w;
    const float* __restrict__ psi_in;
    float* __restrict__ psi_out;
    const double* __restrict__ scale_div;
    int n_items, G, Gs, M, B, Lw, LPT, TPW;
    int slot_bytes, sigt_bytes, chunk_cap;
    float c[kMaxPolar], inv_sin[kMaxPolar], wp[kMaxPolar];
};

template <int N> struct VecT;
template <> struct VecT<4> { using type = float4; };
template <> struct VecT<2> { using type = float2; };
template <> struct VecT<1> { using type = float; };

template <int N>
__device__ __forceinline__ void vload(float (&dst)[N], const float* p)
{
    using V = typename VecT<N>::type;
    const V v = *reinterpret_cast<const V*>(p);
    memcpy(dst, &v, sizeof(V));
}
template <int N>
__device__ __forceinline__ void vstore(float* p, const float (&src)[N])
{
    using V = typename VecT<N>::type;
    V v;
    memcpy(&v, src, sizeof(V));
    *reinterpret_cast<V*>(p) = v;
}

__device__ __forceinline__ int pad_up(int x, int a) { return (x + a - 1) / a * a; }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
template <int BYTES>
__device__ __forceinline__ void cp_async_row(void* smem_dst, const void* gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
    else if (BYTES == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int P, int GPL, int EXPM>
__global__ void __launch_bounds__(512, 1) k_sweep_private(const PrivParams prm)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int Gs = prm.Gs, LPT = prm.LPT, B = prm.B;
    float* sigt_s = reinterpret_cast<float*>(smem);
    for (int i = threadIdx.x; i < prm.M * Gs; i += blockDim.x) sigt_s[i] = prm.sigt[i];
    __syncthreads();
    const int slot = lane / LPT, ll = lane - slot * LPT;
    const bool lane_ok = slot < prm.TPW;
    unsigned char* slot_base = smem + prm.sigt_bytes + (size_t)(warp * prm.TPW + (lane_ok ? slot : 0)) * prm.slot_bytes;
    float* q_s = reinterpret_cast<float*>(slot_base);
    float* acc = q_s + prm.Lw * Gs;
    int32_t* trk_s = reinterpret_cast<int32_t*>(acc + prm.Lw * Gs);          // [B] track ids of the slot's swath
    unsigned char* chunk0 = reinterpret_cast<unsigned char*>(trk_s + pad_up(B, 4));
    if (lane_ok)
        for (int i = ll; i < prm.Lw * Gs; i += LPT) acc[i] = 0.f;
    __syncwarp();
    const float inv_f = (float)(1.0 / *prm.scale_div);
    const int g0 = ll * GPL;                 // first group owned by this lane
    const int hdr_regions = 16 + pad_up(2 * (B + 1), 16);
    const float* sigt_lane = sigt_s + g0;
    const float* q_lane = q_s + g0;
    float* acc_lane = acc + g0;

    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(prm.counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= prm.n_items) break;
        const int4 it = prm.items[item];
        const bool active = lane_ok && slot < it.y;
        const int sw = it.x + (active ? slot : 0);
        const int dir = it.z;
        const int64_t tile0 = prm.swath_tile0[sw];
        const int nt = active ? (int)(prm.swath_tile0[sw + 1] - tile0) : 0;
        const int rounds = __reduce_max_sync(0xffffffffu, nt);
        if (active)
            for (int b = ll; b < B; b += LPT) trk_s[b] = prm.swath_track[(size_t)sw * B + b];
        // chunk offsets (16-byte units) of the first two rounds
        uint32_t c_off = 0, c_n16 = 0, n_off = 0, n_n16 = 0;
        if (nt > 0) {
            const int64_t k = tile0 + (dir ? nt - 1 : 0);
            c_off = prm.tile_chunk[k]; c_n16 = prm.tile_chunk[k + 1] - c_off;
        }
        if (nt > 1) {
            const int64_t k = tile0 + (dir ? nt - 2 : 1);
            n_off = prm.tile_chunk[k]; n_n16 = prm.tile_chunk[k + 1] - n_off;
        }
        {   // stage the first chunk
            const uint4* src = reinterpret_cast<const uint4*>(prm.blob) + c_off;
            for (int i = ll; i < (int)c_n16; i += LPT) cp_async16(reinterpret_cast<uint4*>(chunk0) + i, src + i);
            cp_async_commit();
        }
        __syncwarp();

        for (int round = 0; round < rounds; ++round) {
            const bool has = round < nt;   // nt == 0 for inactive lanes
            unsigned char* chunk = chunk0 + (round & 1) * prm.chunk_cap;
            cp_async_wait<0>();
            __syncwarp();
            int L = 0, nseg = 0;
            if (has) {
                const uint4 h = *reinterpret_cast<const uint4*>(chunk);
                L = (int)h.x; nseg = (int)h.z;
            }
            const uint16_t* seg_start = reinterpret_cast<const uint16_t*>(chunk + 16);
            const uint32_t* regions = reinterpret_cast<const uint32_t*>(chunk + hdr_regions);
            const float* seg_len = reinterpret_cast<const float*>(regions + pad_up(L, 4));
            const uint16_t* seg_im = reinterpret_cast<const uint16_t*>(seg_len + pad_up(nseg, 4));
            // ---- async: q rows of this tile's regions, then the next tile's chunk ----
            for (int l = 0; l < L; ++l) {
                const uint32_t r = regions[l] & 0x00ffffffu;
                cp_async_row<4 * GPL>(q_s + l * Gs + g0, prm.q + (size_t)r * Gs + g0);
            }
            cp_async_commit();
            if (round + 1 < nt) {
                const uint4* src = reinterpret_cast<const uint4*>(prm.blob) + n_off;
                uint4* dst = reinterpret_cast<uint4*>(chunk0 + ((round + 1) & 1) * prm.chunk_cap);
                for (int i = ll; i < (int)n_n16; i += LPT) cp_async16(dst + i, src + i);
            }
            cp_async_commit();
            if (round + 2 < nt) {
                const int64_t k = tile0 + (dir ? nt - 3 - round : round + 2);
                n_off = prm.tile_chunk[k]; n_n16 = prm.tile_chunk[k + 1] - n_off;
            }
            // ---- psi of the first track while the q rows land ----
            float psin[P][GPL];
            float wt_n = 0.f;
            int t_n = has ? trk_s[0] : -1;
            const float* psi_src = round == 0 ? prm.psi_in : prm.psi_out;
            if (t_n >= 0) {
                const size_t at = ((size_t)(2 * t_n + dir) * P) * Gs + g0;
#pragma unroll
                for (int p = 0; p < P; ++p) vload<GPL>(psin[p], psi_src + at + (size_t)p * Gs);
                wt_n = prm.trk_w[t_n];
            }
            cp_async_wait<1>();
            __syncwarp();
            // ---- the B tracks of the swath, one after the other, through this tile ----
            for (int b = 0; b < B; ++b) {
                const int t = t_n;
                float psi[P][GPL], wpt[P];
                int s0 = 0, cnt = 0;
                size_t psi_at = 0;
                if (t >= 0) {
                    s0 = seg_start[b];
                    cnt = seg_start[b + 1] - s0;
                    psi_at = ((size_t)(2 * t + dir) * P) * Gs + g0;
                    const float f = round == 0 ? inv_f : 1.f;
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        wpt[p] = wt_n * prm.wp[p];
#pragma unroll
                        for (int j = 0; j < GPL; ++j) psi[p][j] = psin[p][j] * f;
                    }
                }
                // prefetch the next track's psi (consumed at the next b)
                t_n = (has && b + 1 < B) ? trk_s[b + 1] : -1;
                if (t_n >= 0) {
                    const size_t at = ((size_t)(2 * t_n + dir) * P) * Gs + g0;
#pragma unroll
                    for (int p = 0; p < P; ++p) vload<GPL>(psin[p], psi_src + at + (size_t)p * Gs);
                    wt_n = prm.trk_w[t_n];
                }
                const int steps = __reduce_max_sync(0xffffffffu, cnt);
                // software pipeline: segment record, q row and Sigma_t row of step i+1 are loaded during step i
                const int kstep = dir ? -1 : 1;
                int k = dir ? s0 + cnt - 1 : s0;
                float s_n = 0.f, qn[GPL], stn[GPL];
                int row_n = 0;
                if (cnt > 0) {
                    s_n = seg_len[k];
                    const uint32_t im = seg_im[k];
                    row_n = (int)(im & 0xffu) * Gs;
                    vload<GPL>(qn, q_lane + row_n);
                    vload<GPL>(stn, sigt_lane + (im >> 8) * Gs);
                }
                for (int i = 0; i < steps; ++i) {
                    if (i < cnt) {
                        const float s = s_n;
                        const int row = row_n;
                        float qv[GPL], st[GPL], a4[GPL];
#pragma unroll
                        for (int j = 0; j < GPL; ++j) { qv[j] = qn[j]; st[j] = stn[j]; }
                        vload<GPL>(a4, acc_lane + row);
                        if (i + 1 < cnt) {
                            k += kstep;
                            s_n = seg_len[k];
                            const uint32_t im = seg_im[k];
                            row_n = (int)(im & 0xffu) * Gs;
                            vload<GPL>(qn, q_lane + row_n);
                            vload<GPL>(stn, sigt_lane + (im >> 8) * Gs);
                        }
                        float sc[P];
#pragma unroll
                        for (int p = 0; p < P; ++p) sc[p] = s * (EXPM == 0 ? prm.c[p] : -prm.inv_sin[p]);
#pragma unroll
                        for (int j = 0; j < GPL; ++j) {
#pragma unroll
                            for (int p = 0; p < P; ++p) {
                                const float d = psi[p][j] - qv[j];
                                float delta;
                                if (EXPM == 0) delta = fmaf(-d, ex2_approx(st[j] * sc[p]), d);
                                else delta = d * (-expm1f(st[j] * sc[p]));
                                psi[p][j] -= delta;
                                a4[j] = fmaf(wpt[p], delta, a4[j]);
                            }
                        }
                        vstore<GPL>(acc_lane + row, a4);
                    }
                }
                if (t >= 0) {
#pragma unroll
                    for (int p = 0; p < P; ++p) vstore<GPL>(prm.psi_out + psi_at + (size_t)p * Gs, psi[p]);
                }
            }
            __syncwarp();
            // ---- flush the private window: one FP64 RED per (region, group) of the tile ----
            for (int l = 0; l < L; ++l) {
                const uint32_t r = regions[l] & 0x00ffffffu;
#pragma unroll
                for (int j = 0; j < GPL; ++j) {
                    const int g = ll + LPT * j;              // transposed mapping: a RED covers LPT consecutive doubles
                    if (g < prm.G) {
                        const float v = acc[l * Gs + g];
                        acc[l * Gs + g] = 0.f;
                        atomicAdd(prm.tally + (size_t)r * Gs + g, (double)v);
                    }
                }
            }
            __syncwarp();
        }
        cp_async_wait<0>();
        __syncwarp();
    }
}

} // namespace ndk

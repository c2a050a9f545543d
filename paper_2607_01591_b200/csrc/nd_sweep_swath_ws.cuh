// nd_sweep_swath_ws.cuh -- row A2, warp-specialised variant of k_sweep_swath (ND_SWEEP_SWATH_WS).
//
// profiles/r01d_swath_phases.md: in k_sweep_swath a warp is inside the segment loop for less than half of its cycles;
// the tally flush and the block barriers around it take 36 %.  Here the block is split into
//   * COMPUTE warps (warps 0 .. ncw-1): nothing but the segment loop.  psi in registers along the whole track, one tile
//     after the other, delta rows into one of TWO delta buffers;
//   * SERVICE warps (the last nsw warps): chunk TMA, q-row gathers and the tally flush, one tile behind the compute
//     warps.
// There is no block barrier in the tile loop: the two roles meet at mbarriers --
//   cfull[4]   chunk of tile s landed           (TMA complete_tx, armed by the issuing service thread)
//   qfull[2]   q rows of tile s landed          (cp.async.mbarrier.arrive.noinc by every service thread)
//   dfull[2]   all compute warps finished tile s (lane 0 of every compute warp arrives)
//   dempty[2]  the flush of tile s is over       (lane 0 of every service warp arrives)
// so a compute warp that finishes a tile early simply starts the next one (it can run one tile ahead of the flush).
// Same chunk stream, same segment loop, same results as k_sweep_swath.  Work items are dealt round-robin (item =
// blockIdx.x + n * gridDim.x over the cost-sorted list), so both roles can walk the same sequence without talking.
#pragma once
#include "nd_sweep_swath.cuh"

namespace ndk {

__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// arrive on `bar` once all cp.async operations this thread has issued so far are complete (count pre-charged at init)
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint64_t* bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

struct SwathWsParams {
    SwathParams base;
    int ncw, nsw;   // compute warps, service warps (blockDim.x = 32 * (ncw + nsw))
};

template <int P>
__global__ void __launch_bounds__(384, 2) k_sweep_swath_ws(const SwathWsParams wp)
{
    const SwathParams& prm = wp.base;
    extern __shared__ __align__(128) unsigned char smem_ws[];
    unsigned char* const smem = smem_ws;
    uint64_t* cfull = reinterpret_cast<uint64_t*>(smem);        // [4]
    uint64_t* qfull = cfull + 4;                                 // [2]
    uint64_t* dfull = cfull + 6;                                 // [2]
    uint64_t* dempty = cfull + 8;                                // [2]   (80 bytes of barriers; off_sigt >= 128)
    const int tid = threadIdx.x;
    const int Gs = prm.Gs, row_bytes = 4 * Gs, line = prm.NC * row_bytes;
    unsigned char* sigt_s = smem + prm.off_sigt;
    unsigned char* q_s = smem + prm.off_q;
    unsigned char* dbuf_s = smem + prm.off_dbuf;
    unsigned char* chunk_s = smem + prm.off_chunk;
    const int q_buf_bytes = prm.Lmax * line;
    const int dbuf_bytes = (prm.NT / prm.NC) * prm.Kmax * line;
    const int nq = Gs >> 2;
    const int n_compute = 32 * wp.ncw, n_service = 32 * wp.nsw;

    if (tid == 0) {
        for (int i = 0; i < 4; ++i) mbar_init(cfull + i, 1);
        for (int i = 0; i < 2; ++i) { mbar_init(qfull + i, n_service); mbar_init(dfull + i, wp.ncw); mbar_init(dempty + i, wp.nsw); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < prm.M * prm.NC * nq; i += blockDim.x) {
        const int m = i / (prm.NC * nq), rem = i - m * (prm.NC * nq), piece = rem % nq;
        *reinterpret_cast<float4*>(sigt_s + (size_t)m * line + rem * 16) = *reinterpret_cast<const float4*>(prm.sigt + (size_t)m * Gs + piece * 4);
    }
    __syncthreads();

    uint32_t seq = 0;   // tiles this block has been through: buffers and barrier parities follow it (both roles count alike)
    if (tid < n_compute) {
        // =========================================== COMPUTE ===========================================
        int slot = tid / prm.LPT, ll = tid - slot * prm.LPT;
        const bool lane_ok = slot < prm.NT;
        if (!lane_ok) { slot = prm.NT - 1; ll = prm.LPT - 1; }
        const int sub = slot % prm.NC;
        const int lane_off = sub * row_bytes + ll * 16;
        const unsigned char* sigt_lane = sigt_s + lane_off;
        const int d_slot_off = (slot / prm.NC) * prm.Kmax * line + lane_off;
        const float inv_f = (float)(1.0 / *prm.scale_div);
        const int g0 = ll * 4;
        for (int item = blockIdx.x; item < prm.n_items; item += gridDim.x) {
            const int4 it = prm.items[item];
            const int sw = it.x, dir = it.y;
            const int nt = (int)(prm.swath_tile0[sw + 1] - prm.swath_tile0[sw]);
            const int t = prm.swath_track[(size_t)sw * prm.NT + slot];
            float psi[P][4], wpt[P];
            size_t psi_at = 0;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                wpt[p] = 0.f;
#pragma unroll
                for (int j = 0; j < 4; ++j) psi[p][j] = 0.f;
            }
            if (t >= 0) {
                psi_at = ((size_t)(2 * t + dir) * P) * Gs + g0;
                const float wt = prm.trk_w[t];
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const float4 v = *reinterpret_cast<const float4*>(prm.psi_in + psi_at + (size_t)p * Gs);
                    psi[p][0] = v.x * inv_f; psi[p][1] = v.y * inv_f; psi[p][2] = v.z * inv_f; psi[p][3] = v.w * inv_f;
                    wpt[p] = wt * prm.wp[p];
                }
            }
            for (int k = 0; k < nt; ++k) {
                const uint32_t s = seq + k, b = s & 1u, n = s >> 1;
                mbar_wait(cfull + (s & 3u), (s >> 2) & 1u);   // records of this tile
                mbar_wait(qfull + b, n & 1u);                  // its q rows
                mbar_wait(dempty + b, (n & 1u) ^ 1u);          // the flush of tile s-2 has left this delta buffer
                const SwathChunk ch = decode_chunk(chunk_s + (size_t)(s & 3u) * prm.chunk_cap);
                unsigned char* dbuf = dbuf_s + (size_t)b * dbuf_bytes;
                int s0 = 0, cnt = 0;
                if (t >= 0) { s0 = ch.slot_start[slot]; cnt = ch.slot_start[slot + 1] - s0; }
                const int steps = __reduce_max_sync(0xffffffffu, cnt);
                const unsigned char* q_lane = q_s + (size_t)b * q_buf_bytes + lane_off;
                const int jstep = dir ? -1 : 1;
                const int j_c = dir ? cnt - 1 : 0;
                segment_loop<P, 0>(psi, wpt, prm, ch.rec + s0 + j_c, jstep, cnt, steps, lane_ok, q_lane, sigt_lane,
                                   dbuf + d_slot_off + j_c * line, jstep * line);
                __syncwarp();
                if ((tid & 31) == 0) mbar_arrive(dfull + b);    // release: this warp's delta rows of tile s are written
            }
            seq += (uint32_t)nt;
            if (t >= 0 && lane_ok) {
#pragma unroll
                for (int p = 0; p < P; ++p)
                    *reinterpret_cast<float4*>(prm.psi_out + psi_at + (size_t)p * Gs) = make_float4(psi[p][0], psi[p][1], psi[p][2], psi[p][3]);
            }
        }
        return;
    }
    // =============================================== SERVICE ===============================================
    const int ftid = tid - n_compute;
    const bool leader = ftid == 0;
    const int f_qd = ftid % nq, f_l0 = ftid / nq, f_lstep = n_service / nq;
    const bool f_ok = f_l0 < f_lstep;
    for (int item = blockIdx.x; item < prm.n_items; item += gridDim.x) {
        const int4 it = prm.items[item];
        const int sw = it.x, dir = it.y;
        const int64_t tile0 = prm.swath_tile0[sw];
        const int nt = (int)(prm.swath_tile0[sw + 1] - tile0);
        auto issue_chunk = [&](int k) {   // leader only
            const int64_t ti = tile0 + (dir ? nt - 1 - k : k);
            const uint32_t o0 = prm.tile_chunk[ti], o1 = prm.tile_chunk[ti + 1];
            const uint32_t bytes = (o1 - o0) * 16u, cb = (seq + k) & 3u;
            mbar_expect_tx(cfull + cb, bytes);
            tma_load_1d(chunk_s + (size_t)cb * prm.chunk_cap, prm.blob + (size_t)o0 * 16, bytes, cfull + cb);
        };
        auto issue_q_rows = [&](int k) {   // every service thread: q rows of tile k -> q buffer (seq+k)&1, then arrive
            const uint32_t s = seq + k;
            mbar_wait(cfull + (s & 3u), (s >> 2) & 1u);
            const unsigned char* cb = chunk_s + (size_t)(s & 3u) * prm.chunk_cap;
            const uint4 h = *reinterpret_cast<const uint4*>(cb);
            const int L = (int)(h.x & 0xffffu);
            const uint32_t* regions = reinterpret_cast<const uint32_t*>(cb + 16 * (h.y & 0xffffu));
            const uint32_t qb = smem_u32(q_s + (size_t)(s & 1u) * q_buf_bytes);
            const int per_row = prm.NC * nq;
            for (int i = ftid; i < L * per_row; i += n_service) {
                const int l = (int)fastdiv((uint32_t)i, prm.magic_per_row), rem = i - l * per_row;
                const int piece = rem - (int)fastdiv((uint32_t)rem, prm.magic_nq) * nq;
                cp_async_16(qb + l * line + rem * 16, prm.q + (size_t)regions[l] * Gs + piece * 4);
            }
            cp_async_mbar_arrive_noinc(qfull + (s & 1u));
        };
        // prologue: the chunks of the first four tiles in flight, the q rows of the first two
        if (leader)
            for (int k = 0; k < nt && k < 4; ++k) issue_chunk(k);
        for (int k = 0; k < nt && k < 2; ++k) issue_q_rows(k);
        for (int k = 0; k < nt; ++k) {
            const uint32_t s = seq + k, b = s & 1u, n = s >> 1;
            mbar_wait(cfull + (s & 3u), (s >> 2) & 1u);
            mbar_wait(dfull + b, n & 1u);                    // every compute warp is through tile k: q[b] and the records are free
            if (k + 2 < nt) issue_q_rows(k + 2);             // into q[b], in flight during the flush
            const SwathChunk ch = decode_chunk(chunk_s + (size_t)(s & 3u) * prm.chunk_cap);
            const unsigned char* dbuf = dbuf_s + (size_t)b * dbuf_bytes;
            if (f_ok) {
                for (int l = f_l0; l < ch.L; l += f_lstep) {
                    const int e0 = ch.csr_off[l], e1 = ch.csr_off[l + 1];
                    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                    for (int e = e0; e < e1; ++e) {
                        const float4 x = *reinterpret_cast<const float4*>(dbuf + (size_t)ch.csr_idx[e] * row_bytes + f_qd * 16);
                        v.x += x.x; v.y += x.y; v.z += x.z; v.w += x.w;
                    }
                    double* tp = prm.tally + (size_t)ch.regions[l] * Gs + f_qd * 4;
                    const int gq = f_qd * 4;
                    atomicAdd(tp, (double)v.x);
                    if (gq + 1 < prm.G) atomicAdd(tp + 1, (double)v.y);
                    if (gq + 2 < prm.G) atomicAdd(tp + 2, (double)v.z);
                    if (gq + 3 < prm.G) atomicAdd(tp + 3, (double)v.w);
                }
            }
            __syncwarp();
            if ((ftid & 31) == 0) mbar_arrive(dempty + b);   // this warp no longer reads the delta buffer / the chunk's CSR
            if (leader) {
                mbar_wait(dempty + b, n & 1u);               // ALL service warps are out of chunk k before its buffer is refilled
                if (k + 4 < nt) issue_chunk(k + 4);
            }
        }
        seq += (uint32_t)nt;
    }
}

} // namespace ndk

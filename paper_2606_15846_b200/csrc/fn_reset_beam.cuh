// fn_reset_beam.cuh -- S5 + S6 in ONE launch: reset of the listed envs and the recompute of their beams
// ("resets ... recompute only the affected environments").
//
// As two kernels (reset_kernel, then beam_kernel over the list) the reset path of a step costs two launch
// latencies and, in the reset kernel, a chain of dependent L2 reads of the map (32 start-pose attempts,
// window rows, exact polygon test, goal attempts): ~30 us of a ~100 us step at 4096 envs although only
// ~5 % of the envs are reset.  Here every CTA stages the packed map once (before the dependency wait,
// like beam_kernel), owns the listed envs li = blockIdx.x + k * gridDim.x, resets them from the SHARED
// copy of the map (reset_env<true>: the same code as reset_kernel, so the accepted poses are identical),
// and then casts the beams of its own envs.  No CTA reads another CTA's poses, so a block barrier is the
// only synchronisation.  Used for fn_reset(mask = NULL), the step's done list, when the map is staged in
// shared memory; a caller's mask (long lists: two reset warps per CTA and no balancing of the beams across
// CTAs lose there) and maps read through L2 take the two kernels.
// A reset prepared by the step before (fn_sim_prepare_reset) takes prepared_reset_kernel below instead.
#pragma once
#include "fn_beam.cuh"
#include "fn_env.cuh"

namespace fn {

constexpr int kFusedResetWarps = 2;      // warps of a CTA that run resets (each needs a ColScratch)
constexpr int kFusedPoseSlots = 8;       // sensing poses of a CTA's first envs are kept in shared memory too
constexpr int kFusedThreads = 512;       // two CTAs per SM like beam_kernel (one CTA of 1024 threads measured the same)

__host__ __device__ inline size_t fused_scratch_offset(int B, int mapWords) {      // 32-byte aligned (BeamPose)
    return (((size_t)B * sizeof(double2) + (size_t)mapWords * 4u) + 31u) & ~(size_t)31u;
}
__host__ __device__ inline size_t fused_smem_bytes(int B, int mapWords, int V) {
    return fused_scratch_offset(B, mapWords) + kFusedPoseSlots * sizeof(BeamPose) + kFusedResetWarps * col_scratch_bytes(V);
}

template <bool kAux>
__global__ void __launch_bounds__(kFusedThreads, 2) reset_beam_kernel(const __grid_constant__ ResetArgs ra, const __grid_constant__ BeamArgs a) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B, V = a.robot.V;
    const int rowWords = (a.map.H + 2 * kLineGuard) * a.map.strideR;
    const int mapWords = rowWords + (a.map.W + 2 * kLineGuard) * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    BeamPose* s_pose = reinterpret_cast<BeamPose*>(smem_raw + fused_scratch_offset(B, mapWords));
    uint8_t* s_scr = reinterpret_cast<uint8_t*>(s_pose + kFusedPoseSlots);
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __shared__ __align__(8) unsigned long long s_mbar;
    __shared__ __align__(16) typename std::conditional<!kAux, FastShared<kFusedThreads / 32>, int>::type s_fast;
    stage_beam_constants(a, s_tab, s_map, mapWords, true, &s_mbar);
    ColScratch scratch = col_scratch(s_scr + (size_t)(wib < kFusedResetWarps ? wib : 0) * col_scratch_bytes(V), V);
    if (wib < kFusedResetWarps)
        for (int k = lane; k < V; k += 32) { scratch.verts[k] = a.robot.verts[k]; scratch.nxt[k] = a.robot.nxt[k]; }
    __syncthreads();
    griddep_wait();                                                // the list comes from the kernel before
    griddep_launch_dependents();
    const int* rlist = ra.list;
    const int* rcount = ra.count_dev;
    if (ra.list_par_dev) { const int q = *ra.list_par_dev ^ 1; rlist += (size_t)q * ra.n; rcount += q; }
    const int count = *rcount;
    // this CTA's envs: list entries blockIdx.x, blockIdx.x + gridDim.x, ...
    const int m_loc = count > (int)blockIdx.x ? (count - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    if (m_loc == 0) return;                                        // (uniform over the CTA)

    // ---- phase 1: resets, from the shared copy of the map
    if (wib < kFusedResetWarps) {
        MapDev ms = ra.map;
        ms.row = s_map;
        ms.col = s_map + rowWords;
        for (int k = wib; k < m_loc; k += kFusedResetWarps)
            reset_env<true>(ra, ms, scratch, rlist[blockIdx.x + k * gridDim.x], lane, k < kFusedPoseSlots ? s_pose + k : nullptr);
        __threadfence_block();                                     // poses: written here, read below by all warps
    }
    __syncthreads();

    // ---- phase 2: the beams of this CTA's envs
    const unsigned long long ring_head = a.ring_obs ? *a.ring_head : 0ull;
    if constexpr (!kAux) {                                         // production path: chunks of one env's beams per warp task
        FastWarp w = fast_warp(a, &s_fast, s_tab, (uint32_t)__cvta_generic_to_shared(s_map));
        const unsigned rounds = ((unsigned)B + 31u) >> 5, ntasks = (unsigned)m_loc * rounds;   // a task = 32 beams of one env
        for (unsigned task = (unsigned)wib; task < ntasks; task += blockDim.x >> 5) {
            const unsigned k = a.inv_rounds ? __umulhi(task, a.inv_rounds) : task / rounds, jb0 = (task - k * rounds) << 5;
            const unsigned e = (unsigned)rlist[blockIdx.x + k * gridDim.x];
            fast_chunk<false>(a, w, k < (unsigned)kFusedPoseSlots ? s_pose + k : a.poses + e, e, jb0, min((unsigned)B, jb0 + 32u), ring_head);
        }
        fast_finish(a, w, ring_head);
    } else {                                                       // instrumented: 32 consecutive (env, beam) pairs per warp task
        BeamMap<SmemSpace> bm;
        bm.base = (uint32_t)__cvta_generic_to_shared(s_map);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = (unsigned)rowWords * 4u; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        const unsigned total = (unsigned)m_loc * (unsigned)B;
        const unsigned ntasks = (total + 31u) >> 5;
        const unsigned long long invB = ~0ull / (unsigned long long)B + 1ull;     // floor(2^64 / B) + 1
        uint32_t words = 0, rays = 0;
        for (unsigned task = (unsigned)wib; task < ntasks; task += blockDim.x >> 5) {
            const unsigned idx = (task << 5) + lane;
            const unsigned k = B > 1 ? (unsigned)__umul64hi((unsigned long long)idx, invB) : idx;      // idx / B
            const unsigned j = idx - k * (unsigned)B;
            if (k < (unsigned)m_loc) {
                const unsigned e = (unsigned)rlist[blockIdx.x + k * gridDim.x];
                const BeamPose* pose = k < (unsigned)kFusedPoseSlots ? s_pose + k : a.poses + e;
                beam_element<SmemSpace, kAux>(a, bm, s_tab, pose, e, j, ring_head, words);
                ++rays;
            }
        }
        for (int o = 16; o > 0; o >>= 1) {
            rays += __shfl_xor_sync(0xffffffffu, rays, o);
            words += __shfl_xor_sync(0xffffffffu, words, o);
        }
        if (lane == 0 && rays) {
            atomicAdd(&a.counters[kRays], (unsigned long long)rays);
            if (a.count_words) atomicAdd(&a.counters[kWords], (unsigned long long)words);
        }
    }
}

// fn_reset(mask = NULL) after a step that prepared the resets (fn_sim_prepare_reset): the new states, goal
// observations and sensing poses of the listed envs already sit in the sim's buffers (pr; a.poses = pr.poses), so
// nothing here depends on anything but the list -- every warp of the grid takes rounds of 32 beams of the listed
// envs (task t = round t % rounds of list entry t / rounds, dealt to the CTAs in turn so that the SMs share every
// env's beams); the tasks after those copy the prepared states into the caller's arrays, 32 envs per warp
// (reset_apply).  No reset warps, no block barrier between resetting and casting.
__global__ void __launch_bounds__(kBeamThreads, 2) prepared_reset_kernel(const __grid_constant__ ResetArgs ra, const __grid_constant__ BeamArgs a,
                                                                        const PreparedReset pr) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B;
    const int mapWords = (a.map.H + 2 * kLineGuard) * a.map.strideR + (a.map.W + 2 * kLineGuard) * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    __shared__ __align__(8) unsigned long long s_mbar;
    __shared__ __align__(16) FastShared<kBeamThreads / 32> s_fast;
    stage_beam_constants(a, s_tab, s_map, mapWords, true, &s_mbar);
    __syncthreads();
    griddep_wait();                                                // the list comes from the step
    griddep_launch_dependents();
    const int* rlist = ra.list;
    const int* rcount = ra.count_dev;
    if (ra.list_par_dev) { const int q = *ra.list_par_dev ^ 1; rlist += (size_t)q * ra.n; rcount += q; }
    const unsigned count = (unsigned)*rcount;
    const unsigned long long ring_head = a.ring_obs ? *a.ring_head : 0ull;
    FastWarp w = fast_warp(a, &s_fast, s_tab, (uint32_t)__cvta_generic_to_shared(s_map));
    const unsigned rounds = ((unsigned)B + 31u) >> 5, ntasks = count * rounds, nall = ntasks + ((count + 31u) >> 5);
    const unsigned lane = threadIdx.x & 31, nwarps = gridDim.x * (blockDim.x >> 5);
    for (unsigned task = blockIdx.x + gridDim.x * (threadIdx.x >> 5); task < nall; task += nwarps) {
        if (task < ntasks) {
            const unsigned k = a.inv_rounds ? __umulhi(task, a.inv_rounds) : task / rounds, jb0 = (task - k * rounds) << 5;
            const unsigned e = (unsigned)rlist[k];
            fast_chunk<false>(a, w, a.poses + e, e, jb0, min((unsigned)B, jb0 + 32u), ring_head);
        } else {
            const unsigned k = ((task - ntasks) << 5) + lane;
            if (k < count) reset_apply(ra, pr, rlist[k]);
        }
    }
    fast_finish(a, w, ring_head);
}

}  // namespace fn

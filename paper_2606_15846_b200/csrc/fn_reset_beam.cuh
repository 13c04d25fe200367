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
// nothing here depends on anything but the list -- the warps of the grid share the rounds of 32 beams of the listed
// envs, and the prepared states are copied into the caller's arrays (reset_apply_*).  No reset warps, no owner CTA.
//
// Its CTAs become resident while the step kernel's last CTAs still cast (PDL), and what they need -- the done list
// and the prepared poses -- is complete since the step's outcome warps finished (tens of us earlier; they count
// themselves in end->outcomes_done).  So the work is done BEFORE the dependency wait, under the step kernel's tail:
// the ranges are held in registers, and only the stores wait for the step to complete (it writes the terminal
// observation into the same rows, reads the sensing poses the copies replace, and advances the ring head).  Nothing
// of the CALLER'S is written before the wait either -- ranges, state planes, goal observation: whatever the caller
// launched between fn_step and fn_reset to read the pre-reset observation completes first (only the sim's own
// episode bookkeeping and counters, which no one else can see before the stream reaches them, go early).  The
// CTAs arrive in the order of their index over ~8 us, as the step's CTAs leave (measured with globaltimer stamps).  Waiting for a flag of the kernel BEFORE this one needs no co-residency: the step's
// warps never wait for anything.
constexpr unsigned kCopyFirstCta = 48u;
__global__ void __launch_bounds__(kBeamThreads, 2) prepared_reset_kernel(const __grid_constant__ ResetArgs ra, const __grid_constant__ BeamArgs a,
                                                                        const PreparedReset pr, const StepEnd* end, const unsigned n_outcome_warps,
                                                                        const unsigned max_spin) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B;
    const int mapWords = (a.map.H + 2 * kLineGuard) * a.map.strideR + (a.map.W + 2 * kLineGuard) * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    __shared__ __align__(8) unsigned long long s_mbar;
    __shared__ __align__(16) FastShared<kBeamThreads / 32> s_fast;
    stage_beam_constants(a, s_tab, s_map, mapWords, true, &s_mbar);
    // The step's outcome warps have all finished?  They do tens of us before this kernel starts; should the flag not
    // arrive within max_spin polls all the same (a debugger, a time-sliced or preempted context), the CTA gives up the
    // head start instead of the process: it waits for the step to COMPLETE first -- list, poses and flags are then
    // final by definition -- and does the same work behind the wait.  No guard that can fire, same results.
    __shared__ int s_early;
    if (threadIdx.x == 0) {
        const volatile unsigned* flag = &end->outcomes_done;
        int ok = max_spin != 0u && *flag >= n_outcome_warps;      // (max_spin = 0: never take the head start -- tests)
        for (unsigned it = 1; it < max_spin && !ok; ++it) {
            __nanosleep(64);
            ok = *flag >= n_outcome_warps;
        }
        s_early = ok;
        __threadfence();
    }
    __syncthreads();
    if (!s_early) griddep_wait();
    // (read past L1: these words were written while this SM may have held older copies of their lines)
    const int q = __ldcg(&end->par_used);
    const int* rlist = ra.list + (size_t)q * ra.n;
    const unsigned count = (unsigned)__ldcg(ra.count_dev + q);
    FastWarp w = fast_warp(a, &s_fast, s_tab, (uint32_t)__cvta_generic_to_shared(s_map));
    const unsigned rounds = ((unsigned)B + 31u) >> 5, ntasks = count * rounds;
    const unsigned lane = threadIdx.x & 31, wib = threadIdx.x >> 5, nw = blockDim.x >> 5, nwarps = gridDim.x * nw;
    // The last warp of every CTA is a service warp (copies), the others take one round each before the wait: round t
    // goes to warp t % 15 of CTA t / 15, so the CTAs that arrive last -- they replace the step's last CTAs, ~8 us
    // after the first -- have nothing to do for lists of the usual length.  The copies go to the service warps of
    // CTAs that arrive early but not first (the first SMs to free are still busy with the step's other CTA).
    const unsigned rw = nw - 1u, cap = gridDim.x * rw;             // warps that take rounds per CTA; rounds taken before the wait
    const bool service = wib == rw;
    const unsigned ngroups = (count + 7u) >> 3;                    // copies: 8 listed envs per service warp
    const unsigned g0 = (blockIdx.x + gridDim.x - min(gridDim.x - 1u, kCopyFirstCta)) % gridDim.x;

    // ---- before the wait: a round with held results, or the copies that touch nothing the step still uses
    HeldRound held;
    held.store = false;
    HeldPose hp;                                                   // (the first group's: longer lists copy the rest after the wait)
    hp.e = -1;
    HeldState hs;                                                  // the caller's arrays are written after the wait only
    hs.e = -1;
    if (service) {
        for (unsigned g = g0; g < ngroups; g += gridDim.x) {
            const unsigned k = (g << 3) + lane;
            if (lane < 8u && k < count) {
                const int e = __ldcg(rlist + k);
                reset_apply_early(ra, pr, e);
                if (g == g0) { hp = reset_pose_held(ra, pr, e); hs = reset_state_held(ra, pr, e); }
            }
        }
    } else {
        const unsigned t = blockIdx.x * rw + wib;
        if (t < ntasks) {
            const unsigned k = a.inv_rounds ? __umulhi(t, a.inv_rounds) : t / rounds, jb0 = (t - k * rounds) << 5;
            const unsigned e = (unsigned)__ldcg(rlist + k);
            held = fast_round_held<true>(a, w, a.poses + e, e, jb0);
            // (the stores after the wait should find their translations: the kernel ends when they have landed)
            if (held.store) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.out_ranges + (held.e * a.out_stride + a.out_off + held.j)));
        }
    }

    griddep_wait();                                                // ---- the step is complete
    griddep_launch_dependents();
    const unsigned long long ring_head = a.ring_obs ? *a.ring_head : 0ull;
    fast_store_held(a, held, ring_head);
    if (service) {
        reset_pose_store(ra, hp);
        reset_state_store(ra, hs);
        for (unsigned g = g0; g < ngroups; g += gridDim.x) {
            const unsigned k = (g << 3) + lane;
            if (lane < 8u && k < count) {
                const int e = rlist[k];
                if (g != g0) reset_state_store(ra, reset_state_held(ra, pr, e));
                reset_apply_late(ra, pr, e, g != g0);
            }
        }
    }
    // what a long list leaves over, shared by all warps in the usual way
    for (unsigned t = cap + blockIdx.x + gridDim.x * wib; t < ntasks; t += nwarps) {
        const unsigned k = a.inv_rounds ? __umulhi(t, a.inv_rounds) : t / rounds, jb0 = (t - k * rounds) << 5;
        const unsigned e = (unsigned)rlist[k];
        fast_chunk<false>(a, w, a.poses + e, e, jb0, min((unsigned)B, jb0 + 32u), ring_head);
    }
    fast_finish(a, w, ring_head);
}

}  // namespace fn

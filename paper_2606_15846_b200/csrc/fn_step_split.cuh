// fn_step_split.cuh -- fn_step with the env step split around the beam kernel.
//
// The beam kernel needs only the new sensing poses, i.e. the MOTION update (S1): ~2 us of dependent work per
// env.  Collision (S3), goal observation, reward and done (S4) and the bookkeeping (done list, ring row,
// episode counters) are the longer half of the env step (~4-5 us, the exact polygon test) and feed nothing
// in the beam kernel.  So fn_step launches
//   env_motion_kernel : S1, stores the state planes 0-5 and the sensing poses;
//   step_beam_kernel  : the beam kernel (same staging, same task scheduling), in which the LAST warp of every
//                       CTA first runs S3 + S4 for the envs the CTA owns (env_outcome, the code of the
//                       single-kernel env step, reading the map from the CTA's shared copy when there is
//                       one) while the other warps already cast beams, and then joins them.
// The outcome half leaves the step's critical path; the ring-advance launch disappears too (the last CTA to
// finish advances the ring head and flips the done-list parity).
#pragma once
#include "fn_beam.cuh"
#include "fn_env.cuh"

namespace fn {

// S1 only: one thread per env (epw envs per warp, see env_step_kernel)
__global__ void __launch_bounds__(kEnvBlock) env_motion_kernel(EnvArgs a, StepEnd* end) {
    griddep_wait();                                                // states / actions come from earlier work
    griddep_launch_dependents();                                   // the beam kernel may start staging the map now
    if (blockIdx.x == 0 && threadIdx.x == 0) { *a.beam_task_counter = 0u; end->outcomes_done = 0u; }
    const int e = blockIdx.x * a.epw + threadIdx.x;
    if ((int)threadIdx.x >= a.epw || e >= a.n) return;
    if (a.eval_outcome != nullptr && a.eval_outcome[e] != 0) return;   // a completed evaluation case is frozen
    const EnvMotion mo = env_motion(a, e);
    env_motion_store<false>(a, a.map, e, mo);
}

__host__ __device__ inline size_t step_split_scratch_offset(size_t beam_smem) { return (beam_smem + 15u) & ~(size_t)15u; }
__host__ __device__ inline size_t step_split_smem_bytes(size_t beam_smem, int V) {
    return step_split_scratch_offset(beam_smem) + col_scratch_bytes(V);
}

// beam_smem = the beam kernel's dynamic shared bytes (beam table [+ packed map]); epc = envs owned per CTA
// kPrep: the outcome warp also runs the reset (reset_env, the code of fn_reset) of every env it reports done, into
// the buffers ra points at (fn_sim_prepare_reset): that chain of dependent map reads then runs under the beam
// casting of the other warps instead of after the step.
template <bool kSmem, bool kAux, bool kCoarse = false, bool kPrep = false>
__global__ void __launch_bounds__(FastShape<kCoarse>::kThreads, FastShape<kCoarse>::kCtas) step_beam_kernel(const __grid_constant__ BeamArgs a, const __grid_constant__ EnvArgs ea, StepEnd* end, int epc, unsigned beam_smem, const __grid_constant__ typename std::conditional<kPrep, ResetArgs, int>::type ra) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B, V = a.robot.V;
    const int rowWords = (a.map.H + 2 * kLineGuard) * a.map.strideR;
    const int mapWords = rowWords + (a.map.W + 2 * kLineGuard) * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, last_warp = (int)(blockDim.x >> 5) - 1;
    __shared__ __align__(8) unsigned long long s_mbar;
    constexpr bool fast = kSmem && !kAux;
    __shared__ __align__(16) typename std::conditional<fast, FastShared<FastShape<kCoarse>::kThreads / 32>, int>::type s_fast;
    stage_beam_constants(a, s_tab, s_map, kCoarse ? staged_words_coarse(a.map) : mapWords, kSmem, &s_mbar);
    const ColScratch scratch = col_scratch(smem_raw + step_split_scratch_offset(beam_smem), V);
    if (wib == last_warp)
        for (int k = lane; k < V; k += 32) { scratch.verts[k] = a.robot.verts[k]; scratch.nxt[k] = a.robot.nxt[k]; }
    __syncthreads();
    griddep_wait();                                                // poses and states come from env_motion_kernel
    griddep_launch_dependents();
    const int n = a.n_all;
    const unsigned total = (unsigned)n * (unsigned)B;
    // ring: the step's own rows sit at head, the pending rows (this observation) at head + n
    unsigned long long head_old = 0ull, head_new = 0ull;
    if (a.ring_obs) { head_old = *a.ring_head; head_new = (head_old + (unsigned long long)n) % a.ring_cap; }

    // ---- S3 + S4 of the envs this CTA owns, on its last warp, while the other warps cast beams
    if (wib == last_warp) {
        MapDev ms = ea.map;
        if (kSmem) { ms.row = s_map; ms.col = s_map + rowWords; }
        const int e0 = (int)blockIdx.x * epc;
        const int m_own = min(max(n - e0, 0), epc);
        for (int base = 0; base < m_own; base += 32) {
            const int e = e0 + base + lane;
            const bool in_range = base + lane < m_own;
            const int el = in_range ? e : n - 1;
            const EnvMotion mo = env_motion_load(ea, el);
            unsigned dm = env_outcome<kSmem>(ea, ms, scratch, e, el, in_range, lane, mo, head_old, false);
            if constexpr (kPrep) {
                for (; dm; dm &= dm - 1u) reset_env<kSmem>(ra, ms, scratch, e0 + base + (__ffs(dm) - 1), lane);
            } else (void)dm;
        }
        if constexpr (kPrep) {                                     // list entries, count and prepared resets, then the flag
            __syncwarp();
            if (lane == 0) {
                end->par_used = *ea.par_dev;
                __threadfence();
                atomicAdd(&end->outcomes_done, 1u);
            }
        }
    }

    // the static part of the beam tasks is shared by the warps that start at once; the outcome warps arrive
    // late and take pool tasks only
    const unsigned warp0 = blockIdx.x * (unsigned)last_warp + (unsigned)wib;
    const unsigned nwarps = gridDim.x * (unsigned)last_warp;
    const unsigned rowBytes = (unsigned)rowWords * 4u;
    if constexpr (fast) {
        FastWarp w = fast_warp(a, &s_fast, s_tab, (uint32_t)__cvta_generic_to_shared(s_map));
        run_fast_tasks<kCoarse>(a, w, nullptr, n, head_new, warp0, nwarps, wib != last_warp);
    } else if (kSmem) {
        BeamMap<SmemSpace> bm;
        bm.base = (uint32_t)__cvta_generic_to_shared(s_map);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = rowBytes; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        run_beam_tasks<SmemSpace, kAux>(a, bm, s_tab, nullptr, n, total, head_new, warp0, nwarps, wib != last_warp);
    } else {
        BeamMap<GlobalSpace> bm;
        bm.base = (unsigned long long)__cvta_generic_to_global(a.map.row);
        bm.H = a.map.H; bm.W = a.map.W; bm.stride4R = a.map.strideR << 2; bm.stride4C = a.map.strideC << 2;
        bm.rowBytes = rowBytes; bm.mapBytes = (unsigned)mapWords * 4u; bm.oob = a.counters + kOobLoads;
        run_beam_tasks<GlobalSpace, kAux>(a, bm, s_tab, nullptr, n, total, head_new, warp0, nwarps, wib != last_warp);
    }

    // ---- the last CTA to finish closes the step: done-list parity, the other list's count, the ring head
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&end->done_ctas, 1u) == gridDim.x - 1u) {
            __threadfence();
            const int p = *ea.par_dev;                             // the list this step filled; the next step fills the other
            ea.done_count[p ^ 1] = 0;
            *const_cast<int*>(ea.par_dev) = p ^ 1;
            if (a.ring_obs) {                                      // (ring_advance_kernel's work)
                unsigned long long* head = const_cast<unsigned long long*>(a.ring_head);
                head[0] = head_new;
                head[1] += (unsigned long long)n;
                head[3] = head[2];                                 // terminal observations: a new batch starts (TerminalDev)
            }
            end->done_ctas = 0u;
        }
    }
}

}  // namespace fn

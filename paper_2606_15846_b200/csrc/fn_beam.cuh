// fn_beam.cuh -- range sensing: exact first-hit distance of each beam on the bit-packed map.
//
// Operation: r = rho * inf{t : cell(o + t d) occupied}, capped at
// r_max, no hit => r_max.  The traversal is an exact grid walk organised by LINES instead of cells:
//   * the beam's dominant axis is "u", the other "w"; the packing whose bits run along u is used
//     (row-packed for |dx| >= |dy|, column-packed otherwise), so the beam stays in one line for
//     M = |du/dw| >= 1 cells before it crosses into the next line;
//   * per line the beam covers the cell span [floor(U_k), floor(U_{k+1})], U_{k+1} = U_k + M, tracked
//     in 32.32 fixed point (exact integer adds; error < 2^-32 * lines, far below the 1e-5 cell margin);
//   * the span's occupancy bits are read as one 64-bit window (two aligned 32-bit loads), funnel-
//     shifted so that bit 0 is the span's first cell, and the first occupied cell is found with one
//     count-leading/trailing-zeros -- no per-cell stepping;
//   * beams running towards lower u read the window downwards and use clz instead of ctz.
#pragma once
#include "fn_common.cuh"

namespace fn {

// Address spaces for the packed map: staged in shared memory, or read through L1/L2.
struct SmemSpace {
    using addr_t = uint32_t;                                     // shared-window byte address
    static __device__ __forceinline__ uint32_t ld(addr_t a) {
        uint32_t v;
        asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
        return v;
    }
    static __device__ __forceinline__ addr_t add(addr_t a, int words) { return a + 4u * (uint32_t)words; }
};
struct GlobalSpace {
    using addr_t = const uint32_t*;
    static __device__ __forceinline__ uint32_t ld(addr_t a) { return __ldg(a); }
    static __device__ __forceinline__ addr_t add(addr_t a, int words) { return a + words; }
};

template <class MS>
struct BeamMap {
    typename MS::addr_t row, col;
    int H, W, nwR, nwC, strideR, strideC;
};

constexpr double kFix = 4294967296.0;          // 2^32
constexpr double kMaxSlope = 1048576.0;        // 2^20 cells per line: beyond any map

// One beam.  (ox, oy) origin in cells, (dx, dy) unit direction, T = max range in cells.
// Returns range in metres; *hit = linear cell index, -1 (no hit) or -2 (left the map).
template <class MS, bool kCount>
__device__ __forceinline__ float cast_beam(const BeamMap<MS>& bm, double ox, double oy, double dx,
                                           double dy, double T, float rho, float rmax, int* hit,
                                           uint32_t& words) {
    const int jx = __double2int_rd(ox), iy = __double2int_rd(oy);
    if ((unsigned)jx >= (unsigned)bm.W || (unsigned)iy >= (unsigned)bm.H) { *hit = -2; return 0.0f; }
    {
        uint32_t w0 = MS::ld(MS::add(bm.row, iy * bm.strideR + 1 + (jx >> 5)));
        if (kCount) ++words;
        if ((w0 >> (jx & 31)) & 1u) { *hit = iy * bm.W + jx; return 0.0f; }
    }
    const double adx = fabs(dx), ady = fabs(dy);
    const bool mx = adx >= ady;                                   // dominant axis is x
    const double ou = mx ? ox : oy, ow = mx ? oy : ox;
    const double adu = mx ? adx : ady, adw = mx ? ady : adx;
    const bool fu = (mx ? dx : dy) >= 0.0, fw = (mx ? dy : dx) >= 0.0;
    const int Wu = mx ? bm.W : bm.H, Hw = mx ? bm.H : bm.W;
    const int nw = mx ? bm.nwR : bm.nwC, stride = mx ? bm.strideR : bm.strideC;
    const int l0 = mx ? iy : jx;
    const int Wq = nw * 32;

    // does the beam leave the map before r_max?  (outside = occupied)
    bool exit_hit = false;
    {
        const double lo = T, hi_u = (double)Wu - T, hi_w = (double)Hw - T;
        if (!(ou >= lo && ou < hi_u && ow >= lo && ow < hi_w)) {  // the r_max disc is not inside the map
            const double tu = (fu ? (double)Wu - ou : ou) / adu;
            const double tw = adw > 0.0 ? (fw ? (double)Hw - ow : ow) / adw : INFINITY;
            const double te = fmin(tu, tw);
            if (te < T) { T = te; exit_hit = true; }
        }
    }
    const double M = (adw * kMaxSlope > adu) ? adu / adw : kMaxSlope;
    const double q0 = fu ? ou : (double)Wq - ou;                  // forward coordinate along u
    const double f = fw ? (double)(l0 + 1) - ow : ow - (double)l0;
    int lend = __double2int_rd(fw ? ow + T * adw : ow - T * adw);
    lend = max(0, min(Hw - 1, lend));
    const int kend = abs(lend - l0);
    const long long Q0 = __double2ll_rd(q0 * kFix);
    long long Qn = __double2ll_rd((q0 + f * M) * kFix);           // U_1
    const long long Mf = __double2ll_rd(M * kFix);
    const long long Qend = __double2ll_rd((q0 + T * adu) * kFix);
    const int cend = min((int)(Qend >> 32), fu ? Wu - 1 : Wq - 1);

    // word addressing along the line: forward beams read words j, j+1 upwards from the first data
    // word; backward beams read words downwards from the last data word (mirrored coordinate).
    const int wdir = fu ? 1 : -1;
    typename MS::addr_t wbase = MS::add(mx ? bm.row : bm.col, l0 * stride + (fu ? 1 : nw));
    const int lstep = fw ? stride : -stride;

    int c0 = (int)(Q0 >> 32);
    int rem = kend;
    bool found = false;
    long long qe = 0;
    int cq = 0;
    for (;;) {
        const int c1 = (int)(Qn >> 32);
        typename MS::addr_t a = MS::add(wbase, wdir * (c0 >> 5));
        const uint32_t A = MS::ld(a), Bw = MS::ld(MS::add(a, wdir));
        if (kCount) words += 2;
        const int s = c0 & 31;
        const int k = fu ? __clz(__brev(__funnelshift_r(A, Bw, s))) : __clz(__funnelshift_l(Bw, A, s));
        if (k <= c1 - c0) {
            if (k < 32) {                                         // first occupied cell of this span
                cq = c0 + k;
                qe = (k == 0 && rem != kend) ? Qn - Mf : ((long long)cq << 32);
                found = true;
                break;
            }
            // span longer than one window and nothing in its first 32 cells: scan on
            const int cl = min(c1, cend);
            for (int cc = c0 + 32; cc <= cl && !found; cc += 32) {
                typename MS::addr_t a2 = MS::add(wbase, wdir * (cc >> 5));
                const uint32_t A2 = MS::ld(a2), B2 = MS::ld(MS::add(a2, wdir));
                if (kCount) words += 2;
                const int s2 = cc & 31;
                const int k2 = fu ? __clz(__brev(__funnelshift_r(A2, B2, s2))) : __clz(__funnelshift_l(B2, A2, s2));
                if (k2 < 32 && cc + k2 <= cl) { cq = cc + k2; qe = (long long)cq << 32; found = true; }
            }
            if (found) break;
        }
        if (rem == 0) break;
        --rem;
        c0 = c1;
        Qn += Mf;
        wbase = MS::add(wbase, lstep);
    }
    if (found && qe < Qend) {
        const int cu = fu ? cq : Wq - 1 - cq;
        const int line = l0 + (fw ? (kend - rem) : -(kend - rem));
        *hit = mx ? line * bm.W + cu : cu * bm.W + line;
        const long long dq = qe - Q0;
        const float t = (float)(dq > 0 ? dq : 0) * (float)(rho / (adu * kFix));
        return t;
    }
    if (exit_hit) { *hit = -2; return (float)(T * (double)rho); }
    *hit = -1;
    return rmax;
}

struct BeamArgs {
    MapDev map;
    RobotDev robot;
    const PoseD* poses;          // [N]
    const int* list;             // compacted env indices or NULL (= all envs)
    const int* count_dev;        // number of listed envs (device) or NULL
    int n_all;                   // number of envs when list == NULL
    float* out_ranges;           // [N][B]
    int* out_hit;                // [N][B] or NULL
    float* ring_obs;             // ring base or NULL: also write ranges into the env's pending ring row
    unsigned long long ring_cap, ring_head;   // pending row of env e = (ring_head + e) % ring_cap
    int ring_row;                // floats per ring row
    unsigned long long* counters;
};

// Persistent kernel: each CTA stages both packed copies of the map and the beam table in shared
// memory (kSmem) or reads the map through L1/L2 (global path), then its warps take 32 consecutive
// (env, beam) pairs at a time: adjacent lanes = adjacent beams of one env, so a warp's loads mostly hit
// the same or neighbouring words (broadcast) and its lanes run similar trip counts.
template <bool kSmem, bool kCount>
__global__ void __launch_bounds__(512, 2) beam_kernel(BeamArgs a) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B;
    const int rowWords = a.map.H * a.map.strideR, colWords = a.map.W * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    for (int i = threadIdx.x; i < B; i += blockDim.x) s_tab[i] = a.robot.beam_cs[i];
    if (kSmem) {
        const uint4* src = reinterpret_cast<const uint4*>(a.map.row);      // row and col are contiguous
        uint4* dst = reinterpret_cast<uint4*>(s_map);
        const int n4 = (rowWords + colWords + 3) / 4;
        for (int i = threadIdx.x; i < n4; i += blockDim.x) dst[i] = __ldg(src + i);
    }
    __syncthreads();

    using MS = typename std::conditional<kSmem, SmemSpace, GlobalSpace>::type;
    BeamMap<MS> bm;
    if constexpr (kSmem) {
        bm.row = (uint32_t)__cvta_generic_to_shared(s_map);
        bm.col = bm.row + 4u * (uint32_t)rowWords;
    } else {
        bm.row = a.map.row;
        bm.col = a.map.col;
    }
    bm.H = a.map.H; bm.W = a.map.W; bm.nwR = a.map.nwR; bm.nwC = a.map.nwC;
    bm.strideR = a.map.strideR; bm.strideC = a.map.strideC;

    const int n_env = a.count_dev ? *a.count_dev : a.n_all;
    const long long total = (long long)n_env * B;
    const int lane = threadIdx.x & 31;
    const int warps_per_cta = blockDim.x >> 5;
    const long long warp0 = (long long)blockIdx.x * warps_per_cta + (threadIdx.x >> 5);
    const long long nwarps = (long long)gridDim.x * warps_per_cta;
    uint32_t words = 0, rays = 0;
    for (long long task = warp0; task * 32 < total; task += nwarps) {
        const long long idx = task * 32 + lane;
        if (idx < total) {
            const int le = (int)(idx / B), j = (int)(idx - (long long)le * B);
            const int e = a.list ? a.list[le] : le;
            const PoseD p = a.poses[e];
            const double2 cs = s_tab[j];
            const double dx = p.c * cs.x - p.s * cs.y, dy = p.s * cs.x + p.c * cs.y;
            int hit;
            const float r = cast_beam<MS, kCount>(bm, p.ox, p.oy, dx, dy, a.robot.T, a.map.rho,
                                                  a.robot.rmax, &hit, words);
            const size_t o = (size_t)e * B + j;
            a.out_ranges[o] = r;
            if (a.out_hit) a.out_hit[o] = hit;
            if (a.ring_obs) {
                const unsigned long long slot = (a.ring_head + (unsigned long long)e) % a.ring_cap;
                a.ring_obs[slot * a.ring_row + j] = r;
            }
            ++rays;
        }
    }
    // counters: one atomic per warp
    for (int o = 16; o > 0; o >>= 1) {
        rays += __shfl_xor_sync(0xffffffffu, rays, o);
        if (kCount) words += __shfl_xor_sync(0xffffffffu, words, o);
    }
    if (lane == 0) {
        atomicAdd(&a.counters[kRays], (unsigned long long)rays);
        if (kCount) atomicAdd(&a.counters[kWords], (unsigned long long)words);
    }
}

}  // namespace fn

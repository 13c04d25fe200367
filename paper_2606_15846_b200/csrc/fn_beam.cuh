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
#include <type_traits>

namespace fn {

// Address spaces for the packed map: staged in shared memory, or read through L1/L2.
struct SmemSpace {
    using addr_t = uint32_t;                                     // shared-window byte address
    static __device__ __forceinline__ uint32_t ld(addr_t a) {
        uint32_t v;
        asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
        return v;
    }
    static __device__ __forceinline__ addr_t addb(addr_t a, int bytes) { return a + (uint32_t)bytes; }
    static __device__ __forceinline__ int diffb(addr_t a, addr_t b) { return (int)(a - b); }
};
struct GlobalSpace {
    using addr_t = const uint32_t*;
    static __device__ __forceinline__ uint32_t ld(addr_t a) { return __ldg(a); }
    static __device__ __forceinline__ addr_t addb(addr_t a, int bytes) {
        return reinterpret_cast<addr_t>(reinterpret_cast<const char*>(a) + bytes);
    }
    static __device__ __forceinline__ int diffb(addr_t a, addr_t b) {
        return (int)(reinterpret_cast<const char*>(a) - reinterpret_cast<const char*>(b));
    }
};

template <class MS>
struct BeamMap {
    typename MS::addr_t row, col;
    int H, W, nwR, nwC, strideR, strideC;
};

constexpr double kFix = 4294967296.0;          // 2^32
constexpr double kMaxSlope = 1048576.0;        // 2^20 cells per line: beyond any map

__device__ __forceinline__ int bfind32(uint32_t x) {            // msb position, -1 if x == 0 (SASS FLO.U32)
    int r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}
__device__ __forceinline__ int hi32(long long q) { return (int)(q >> 32); }

// The 64-bit occupancy window that starts at forward cell c0 of the current line, normalised so that
// the FIRST cell of the span sits at bit 31 and later cells at lower bits: bfind then names the first
// occupied cell as k = 31 - p.  Both words are at ascending addresses (a, a + 4) in either direction.
template <class MS, bool kFwd, bool kAux>
__device__ __forceinline__ int window_msb(typename MS::addr_t wbase, int c0, uint32_t& words) {
    const int j4 = (c0 >> 5) << 2;
    typename MS::addr_t a = MS::addb(wbase, kFwd ? j4 : -j4);
    const uint32_t L = MS::ld(a), Hh = MS::ld(MS::addb(a, 4));
    if (kAux) words += 2;
    return bfind32(kFwd ? __brev(__funnelshift_r(L, Hh, c0)) : __funnelshift_l(L, Hh, c0));
}

// Walks the lines of one beam.  Returns true with (cq, qe) = forward cell and 32.32 entry coordinate of
// the first occupied cell met, false if the lines up to the end pointer hold none.
template <class MS, bool kFwd, bool kAux>
__device__ __forceinline__ bool walk_lines(typename MS::addr_t wbase, const typename MS::addr_t wend,
                                           const int lstep4, long long Qn, const long long Mf, int c0,
                                           const int cend, int& cq, long long& qe, typename MS::addr_t& wfound,
                                           uint32_t& words) {
    bool first = true;
    for (;;) {
        int p;
        for (;;) {                                               // hot loop: one window per line
            const int c1 = hi32(Qn);
            p = window_msb<MS, kFwd, kAux>(wbase, c0, words);
            if (p >= c0 + 31 - c1) break;                        // first occupied cell lies inside the span
            if (wbase == wend) return false;
            c0 = c1;
            Qn += Mf;
            wbase = MS::addb(wbase, lstep4);
            first = false;
        }
        const int c1 = hi32(Qn);
        if (p >= 0) {
            const int k = 31 - p;
            cq = c0 + k;
            qe = (k == 0 && !first) ? Qn - Mf : ((long long)cq << 32);
            wfound = wbase;
            return true;
        }
        // span longer than one window with an empty first window: scan the rest of it
        const int cl = min(c1, cend);
        for (int cc = c0 + 32; cc <= cl; cc += 32) {
            const int p2 = window_msb<MS, kFwd, kAux>(wbase, cc, words);
            if (p2 >= 0 && cc + 31 - p2 <= cl) {
                cq = cc + 31 - p2;
                qe = (long long)cq << 32;
                wfound = wbase;
                return true;
            }
        }
        if (wbase == wend) return false;
        c0 = c1;
        Qn += Mf;
        wbase = MS::addb(wbase, lstep4);
        first = false;
    }
}

// Hot loop in PTX for the shared-memory map and slopes M < 31 cells per line (span <= 32 cells, so one
// window per line always suffices).  Per line: word address (shr, mad), two ld.shared, funnel shift,
// (brev,) bfind.shiftamt = k, len = c1 - c0, hit = (k <= len) fused with the end-of-lines test into one
// predicate and one branch, then the 64-bit fixed-point add and the line-pointer add: 14 (forward) /
// 13 (backward) instructions.  Unrolled twice with the roles of the (c0, hi(Q)) registers swapped so
// that "c0 := c1" costs nothing.  Returns true when the first occupied cell of the current line's
// window lies inside the beam's span (k = its offset from c0); false when the lines are exhausted.
template <bool kFwd>
__device__ __forceinline__ bool fast_lines_smem(uint32_t& wbase, const uint32_t wend, const int lstep4,
                                                uint32_t& qlo, int& qhi, const uint32_t mlo, const int mhi,
                                                int& c0, int& k) {
    int found, c0o, qho;
#define FN_LINE(RC, RQ, EXIT)                                              \
    "shr.s32 j, " RC ", 5;\n\t"                                            \
    "mad.lo.s32 a, j, %12, %0;\n\t"                                        \
    "ld.shared.u32 L, [a];\n\t"                                            \
    "ld.shared.u32 H, [a+4];\n\t"                                          \
    FN_SHIFT(RC)                                                           \
    "bfind.shiftamt.u32 %4, x;\n\t"                                        \
    "sub.s32 len, " RQ ", " RC ";\n\t"                                     \
    "setp.le.u32 ph, %4, len;\n\t"                                         \
    "setp.eq.or.u32 pe, %0, %8, ph;\n\t"                                   \
    "@pe bra " EXIT ";\n\t"                                                \
    "add.cc.u32 %1, %1, %10;\n\t"                                          \
    "addc.s32 " RC ", " RQ ", %11;\n\t"                                    \
    "add.s32 %0, %0, %9;\n\t"
    if (kFwd) {
#define FN_SHIFT(RC) "shf.r.wrap.b32 x, L, H, " RC ";\n\tbrev.b32 x, x;\n\t"
        asm volatile(
            "{\n\t"
            ".reg .pred ph, pe;\n\t"
            ".reg .b32 j, a, L, H, x, len, rc, rq;\n\t"
            "mov.b32 rc, %2;\n\t"
            "mov.b32 rq, %3;\n\t"
            "FN_LA:\n\t" FN_LINE("rc", "rq", "FN_XA")
            FN_LINE("rq", "rc", "FN_XB")
            "bra FN_LA;\n\t"
            "FN_XA:\n\t"
            "mov.b32 %6, rc;\n\t"
            "mov.b32 %7, rq;\n\t"
            "bra FN_END;\n\t"
            "FN_XB:\n\t"
            "mov.b32 %6, rq;\n\t"
            "mov.b32 %7, rc;\n\t"
            "FN_END:\n\t"
            "selp.s32 %5, 1, 0, ph;\n\t"
            "}"
            : "+r"(wbase), "+r"(qlo), "+r"(c0), "+r"(qhi), "=r"(k), "=r"(found), "=r"(c0o), "=r"(qho)
            : "r"(wend), "r"(lstep4), "r"(mlo), "r"(mhi), "n"(4));
#undef FN_SHIFT
    } else {
#define FN_SHIFT(RC) "shf.l.wrap.b32 x, L, H, " RC ";\n\t"
        asm volatile(
            "{\n\t"
            ".reg .pred ph, pe;\n\t"
            ".reg .b32 j, a, L, H, x, len, rc, rq;\n\t"
            "mov.b32 rc, %2;\n\t"
            "mov.b32 rq, %3;\n\t"
            "FN_LA:\n\t" FN_LINE("rc", "rq", "FN_XA")
            FN_LINE("rq", "rc", "FN_XB")
            "bra FN_LA;\n\t"
            "FN_XA:\n\t"
            "mov.b32 %6, rc;\n\t"
            "mov.b32 %7, rq;\n\t"
            "bra FN_END;\n\t"
            "FN_XB:\n\t"
            "mov.b32 %6, rq;\n\t"
            "mov.b32 %7, rc;\n\t"
            "FN_END:\n\t"
            "selp.s32 %5, 1, 0, ph;\n\t"
            "}"
            : "+r"(wbase), "+r"(qlo), "+r"(c0), "+r"(qhi), "=r"(k), "=r"(found), "=r"(c0o), "=r"(qho)
            : "r"(wend), "r"(lstep4), "r"(mlo), "r"(mhi), "n"(-4));
#undef FN_SHIFT
    }
#undef FN_LINE
    c0 = c0o;
    qhi = qho;
    return found != 0;
}

// One beam.  (ox, oy) origin in cells, (dx, dy) unit direction, T = max range in cells; `inside` = the
// r_max disc around the origin lies inside the map (no exit clipping needed).
// Returns range in metres; *hit = linear cell index, -1 (no hit) or -2 (left the map).
template <class MS, bool kAux>
__device__ __forceinline__ float cast_beam(const BeamMap<MS>& bm, const double ox, const double oy,
                                           const double dx, const double dy, double T, const bool inside,
                                           const float rho, const float rmax, int* hit, uint32_t& words) {
    const int jx = __double2int_rd(ox), iy = __double2int_rd(oy);
    if ((unsigned)jx >= (unsigned)bm.W || (unsigned)iy >= (unsigned)bm.H) { *hit = -2; return 0.0f; }
    {
        const uint32_t w0 = MS::ld(MS::addb(bm.row, (iy * bm.strideR + 1 + (jx >> 5)) << 2));
        if (kAux) ++words;
        if ((w0 >> (jx & 31)) & 1u) { *hit = iy * bm.W + jx; return 0.0f; }
    }
    const bool mx = fabs(dx) >= fabs(dy);                         // dominant axis is x
    const double ou = mx ? ox : oy, ow = mx ? oy : ox;
    const double du = mx ? dx : dy, dw = mx ? dy : dx;
    const double adu = fabs(du), adw = fabs(dw);
    const bool fu = du >= 0.0, fw = dw >= 0.0;
    const int Wu = mx ? bm.W : bm.H, Hw = mx ? bm.H : bm.W;
    const int nw = mx ? bm.nwR : bm.nwC, stride = mx ? bm.strideR : bm.strideC;
    const int l0 = mx ? iy : jx;
    const int Wq = nw << 5;

    // slope M = |du/dw| by one Newton step on the fp32 reciprocal (relative error ~1e-14), capped
    double M;
    {
        const double r0 = (double)__frcp_rn((float)adw);
        const double r1 = r0 * (2.0 - adw * r0);
        M = (adw * kMaxSlope > adu) ? adu * r1 : kMaxSlope;
    }
    bool exit_hit = false;
    if (!inside) {                                                // does the beam leave the map before r_max?
        const double tu = (fu ? (double)Wu - ou : ou) / adu;
        const double tw = adw > 0.0 ? (fw ? (double)Hw - ow : ow) / adw : INFINITY;
        const double te = fmin(tu, tw);
        if (te < T) { T = te; exit_hit = true; }
    }
    const double l0d = (double)l0;
    const double tf = l0d - ow;                                   // in (-1, 0]
    const double f = fw ? tf + 1.0 : -tf;                         // distance to the first line boundary
    const double q0s = (fu ? ou : (double)Wq - ou) * kFix;        // forward coordinate, 32.32 scaled
    const double Ms = M * kFix;
    int lend = __double2int_rd(ow + T * dw);
    lend = max(0, min(Hw - 1, lend));
    const long long Q0 = __double2ll_rd(q0s);
    const long long Qn = __double2ll_rd(q0s + f * Ms);            // U_1
    const long long Mf = __double2ll_rd(Ms);
    const long long Qend = __double2ll_rd(q0s + (T * kFix) * adu);
    const int cend = min(hi32(Qend), fu ? Wu - 1 : Wq - 1);

    const int stride4 = stride << 2;
    const int lstep4 = fw ? stride4 : -stride4;
    typename MS::addr_t line0 = MS::addb(mx ? bm.row : bm.col, l0 * stride4);
    typename MS::addr_t wbase = MS::addb(line0, fu ? 4 : (nw - 1) << 2);
    typename MS::addr_t wend = MS::addb(wbase, (lend - l0) * stride4);
    int cq = 0;
    long long qe = 0;
    typename MS::addr_t wfound = wbase;
    bool found;
    if constexpr (std::is_same<MS, SmemSpace>::value && !kAux) {
        if (hi32(Mf) < 31) {                                      // one window per line always suffices
            uint32_t wb = wbase, qlo = (uint32_t)Qn;
            int qhi = hi32(Qn), c0 = hi32(Q0), k;
            found = fu ? fast_lines_smem<true>(wb, wend, lstep4, qlo, qhi, (uint32_t)Mf, hi32(Mf), c0, k)
                       : fast_lines_smem<false>(wb, wend, lstep4, qlo, qhi, (uint32_t)Mf, hi32(Mf), c0, k);
            cq = c0 + k;
            const long long Qcur = ((long long)qhi << 32) | (long long)qlo;
            qe = (k == 0 && wb != wbase) ? Qcur - Mf : ((long long)cq << 32);
            wfound = wb;
        } else {
            found = fu ? walk_lines<MS, true, kAux>(wbase, wend, lstep4, Qn, Mf, hi32(Q0), cend, cq, qe, wfound, words)
                       : walk_lines<MS, false, kAux>(wbase, wend, lstep4, Qn, Mf, hi32(Q0), cend, cq, qe, wfound, words);
        }
    } else {
        found = fu ? walk_lines<MS, true, kAux>(wbase, wend, lstep4, Qn, Mf, hi32(Q0), cend, cq, qe, wfound, words)
                   : walk_lines<MS, false, kAux>(wbase, wend, lstep4, Qn, Mf, hi32(Q0), cend, cq, qe, wfound, words);
    }
    if (found && qe < Qend) {
        if (kAux) {
            const int cu = fu ? cq : Wq - 1 - cq;
            const int line = l0 + MS::diffb(wfound, wbase) / stride4;
            *hit = mx ? line * bm.W + cu : cu * bm.W + line;
        }
        const long long dq = qe - Q0;
        return (float)(dq > 0 ? dq : 0) * (float)((double)rho / (adu * kFix));
    }
    if (exit_hit) { *hit = -2; return (float)(T * (double)rho); }
    *hit = -1;
    return rmax;
}

struct BeamArgs {
    MapDev map;
    RobotDev robot;
    const PoseD* poses;          // [N]
    const int* pose_inside;      // [N] 1 = the r_max disc around the sensor lies inside the map
    const int* list;             // compacted env indices or NULL (= all envs)
    const int* count_dev;        // number of listed envs (device) or NULL
    int n_all;                   // number of envs when list == NULL
    float* out_ranges;           // [N][B]
    int* out_hit;                // [N][B] or NULL            (kAux only)
    float* ring_obs;             // ring base or NULL: also write ranges into the env's pending ring row
    unsigned long long ring_cap, ring_head;   // pending row of env e = (ring_head + e) % ring_cap
    int ring_row;                // floats per ring row
    int count_words;             // (kAux only)
    unsigned long long* counters;
};

// Persistent kernel: each CTA stages both packed copies of the map and the beam table in shared
// memory (kSmem) or reads the map through L1/L2 (global path), then its warps take 32 consecutive
// (env, beam) pairs at a time: adjacent lanes = adjacent beams of one env, so a warp's loads mostly hit
// the same or neighbouring words (broadcast) and its lanes run similar trip counts.
// kAux = instrumented variant: hit-cell output, map-word counter.
template <bool kSmem, bool kAux>
__global__ void __launch_bounds__(512, 2) beam_kernel(BeamArgs a) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int B = a.robot.B;
    const int n_env = a.count_dev ? *a.count_dev : a.n_all;
    const unsigned total = (unsigned)n_env * (unsigned)B;
    const int warps_per_cta = blockDim.x >> 5;
    if ((unsigned)blockIdx.x * warps_per_cta * 32u >= total) return;      // nothing for this CTA: skip staging
    const int rowWords = a.map.H * a.map.strideR, colWords = a.map.W * a.map.strideC;
    double2* s_tab = reinterpret_cast<double2*>(smem_raw);
    uint32_t* s_map = reinterpret_cast<uint32_t*>(smem_raw + (size_t)B * sizeof(double2));
    for (int i = threadIdx.x; i < B; i += blockDim.x) s_tab[i] = a.robot.beam_cs[i];
    if (kSmem) {
        const uint4* src = reinterpret_cast<const uint4*>(a.map.row);      // row and col are contiguous
        uint4* dst = reinterpret_cast<uint4*>(s_map);
        const int n4 = (rowWords + colWords + 3) / 4;
        int i = threadIdx.x;
        for (; i + 3 * (int)blockDim.x < n4; i += 4 * blockDim.x) {         // 4 loads in flight per thread
            const uint4 v0 = __ldg(src + i), v1 = __ldg(src + i + blockDim.x);
            const uint4 v2 = __ldg(src + i + 2 * blockDim.x), v3 = __ldg(src + i + 3 * blockDim.x);
            dst[i] = v0; dst[i + blockDim.x] = v1; dst[i + 2 * blockDim.x] = v2; dst[i + 3 * blockDim.x] = v3;
        }
        for (; i < n4; i += blockDim.x) dst[i] = __ldg(src + i);
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

    const int lane = threadIdx.x & 31;
    const unsigned warp0 = blockIdx.x * warps_per_cta + (threadIdx.x >> 5);
    const unsigned nwarps = gridDim.x * warps_per_cta;
    const unsigned ntasks = (total + 31u) >> 5;
    uint32_t words = 0, rays = 0;
    for (unsigned task = warp0; task < ntasks; task += nwarps) {
        const unsigned idx0 = task << 5;
        unsigned le = idx0 / (unsigned)B;                              // warp-uniform
        unsigned j = idx0 - le * (unsigned)B + lane;
        while (j >= (unsigned)B) { j -= B; ++le; }
        if (le < (unsigned)n_env) {
            const int e = a.list ? a.list[le] : (int)le;
            const PoseD p = a.poses[e];
            const bool inside = a.pose_inside[e] != 0;
            const double2 cs = s_tab[j];
            const double dx = p.c * cs.x - p.s * cs.y, dy = p.s * cs.x + p.c * cs.y;
            int hit;
            const float r = cast_beam<MS, kAux>(bm, p.ox, p.oy, dx, dy, a.robot.T, inside, a.map.rho,
                                                a.robot.rmax, &hit, words);
            const size_t o = (size_t)e * B + j;
            a.out_ranges[o] = r;
            if (kAux && a.out_hit) a.out_hit[o] = hit;
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
        if (kAux) words += __shfl_xor_sync(0xffffffffu, words, o);
    }
    if (lane == 0) {
        atomicAdd(&a.counters[kRays], (unsigned long long)rays);
        if (kAux && a.count_words) atomicAdd(&a.counters[kWords], (unsigned long long)words);
    }
}

}  // namespace fn

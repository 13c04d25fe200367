// fn_common.cuh -- shared device-side structures and helpers of libflashnav (sm_100a).
// Layouts are described in DESIGN.md "Data layout in HBM".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fn {

constexpr int kMaxVerts = 64;
constexpr int kMaxAttempts = 256;
constexpr int kNCounters = 8;
enum Counter { kRays = 0, kWords = 1, kResets = 2, kResetFail = 3, kNonFinite = 4, kEnvSteps = 5, kOobLoads = 6, kResetsPrepared = 7 };

// Bit-packed map, two orientations.  A "line" is one row of the row-packed copy (bits run along
// columns) or one column of the column-packed copy (bits run along rows).  "Outside the map is
// occupied" is stored physically, so no kernel clips a beam against the map border:
//   * a copy holds L + 4 lines: physical line p = l + 2; lines l = -2, -1, L, L+1 are all ones
//     (l = -1 and L are the frame the beams hit; the outer two are guards for look-ahead reads);
//   * a line is [2 pad words][nw data words][2 pad words] of 32 bits, pads all ones; data bit b of
//     word k is cell 32k + b, bits at or beyond the line's length are ones.  So cell u sits at bit
//     (u + 64) & 31 of physical word (u + 64) >> 5, for u in [-64, 32 nw + 64).
struct MapDev {
    const uint32_t* row;     // [H + 4][strideR]
    const uint32_t* col;     // [W + 4][strideC]   (directly after the row copy)
    int H, W;
    int nwR, nwC;            // data words per line: ceil(W/32), ceil(H/32)
    int strideR, strideC;    // nw + 4
    float rho;               // metres per cell
    double inv_rho;          // 1 / (double)rho
};
constexpr int kCellShift = 64;     // cell u is stored at bit position u + kCellShift of its line
constexpr int kLineGuard = 2;      // physical line = l + kLineGuard
// Coarse level of a copy: line g = the OR of the physical lines 2g and 2g + 1 (a missing odd line counts as
// all ones), same cell -> bit mapping, stored at word offset g * 2 * stride, i.e. at the BIT offset of the fine
// line 2g within its copy: a crossing coordinate D (fn_beam.cuh) addresses the coarse line of a pair and
// the pair's even fine line with the same bits.  One guard pair (all ones) follows the last one.
__host__ __device__ inline size_t coarse_words(int L, int stride) {
    return (size_t)((L + 2 * kLineGuard + 1) / 2 + 1) * 2 * (size_t)stride;
}

// Per-env sensing pose, written by the env/reset/pose kernels, read by the beam kernel.  The beam
// kernel walks along the beam's dominant axis "u" (minor axis "w"); both choices are prepared here:
// o[0]: u = x (row-packed copy, line = row), o[1]: u = y (column-packed copy, line = column).
constexpr double kMagic = 1048576.0;            // 2^20: a double D in [2^20, 2^21) has ulp 2^-32 and its
constexpr unsigned kMagicHi = 0x41300000u;      // high word is exactly kMagicHi + floor(D - 2^20)
struct __align__(16) BeamOrient {
    double ouM;              // origin along u, in cells, + kCellShift + kMagic
    int cu0;                 // floor(origin along u)
    unsigned line_off;       // byte offset of the origin's line from the start of the row copy
    double h;                // 0.5 - frac(origin along w): first line boundary at f = 0.5 +- h
    double ouMS;             // ouM + the BIT offset of the origin's line within its own copy (row / column)
};                           // (h, ouMS) are one 16-byte load of the production beam kernel
struct __align__(32) BeamPose {
    double c, s;             // cos/sin of the heading
    BeamOrient o[2];
    int state;               // 0 = origin in a free cell, 1 = in an occupied cell, 2 = outside the map
    int psi_bits;            // bit pattern of the fp32 heading that (c, s) belong to
    unsigned line_par[2];    // parity of the physical line of the origin in o[0] / o[1] (coarse level: which line of its pair)
};

struct RobotDev {
    const double2* beam_cs;  // [B] (cos, sin) of theta_j + s_psi
    const double2* verts;    // [V] footprint vertices, body frame, metres (components one after the other)
    const int* nxt;          // [V] next vertex within the vertex's component (a union of polygons)
    const double2* samples;  // [n_samples] points inside the footprint (body frame): a cheap one-sided pre-test
    int n_samples;
    int B, V;
    int drive;               // 0 diff, 1 omni
    int A;                   // action dim
    float lim[6];
    float acc[3];            // maximum accelerations a_x, a_y, a_w (+inf = none; reading G2)
    float rmax;              // metres
    double T;                // rmax / rho in cells
    double sx, sy;           // sensor offset, metres (sensor 0)
    int n_sensors;           // range sensors of the robot; poses of sensor k: poses[k * n_envs + e]
    double sxs[4], sys[4];   // their offsets
};

struct TaskDev {
    float goal_tol;
    int max_episode_steps;
    float dmin, dmax;
    float r_success, r_collision, c_progress;
};

struct RegionsDev {
    const int4* rects;       // (row0, col0, h, w)
    int n;
};

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// Programmatic dependent launch (PDL): every kernel of fn_step / fn_reset is launched with the
// programmatic-stream-serialization attribute, so it may become resident while its predecessor in the
// stream still runs.  griddepcontrol.wait blocks until that predecessor has COMPLETED and its memory is
// visible (and, by induction, everything before it); what a kernel does before the wait may only touch
// constants of the map / robot (the beam kernel stages the map there).  launch_dependents, issued
// right after the wait, lets the next kernel's CTAs be scheduled as soon as resources free up.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }

__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// wrap to [-pi, pi)
__device__ __forceinline__ double wrap_pi(double a) {
    const double two_pi = 6.283185307179586476925286766559;
    const double pi = 3.141592653589793238462643383279;
    double r = a - two_pi * floor((a + pi) * 0.15915494309189533576888376337251);   // (a + pi) / (2 pi)
    if (r >= pi) r -= two_pi;
    if (r < -pi) r += two_pi;
    return r;
}

// One word of the packed map.  kS = false: the copy in global memory (read-only path).  kS = true: m.row
// points at a copy staged in shared memory (the fused reset + beam kernel), read with a generic load.
template <bool kS = false>
__device__ __forceinline__ uint32_t map_word(const uint32_t* p) {
    if constexpr (kS) return *p; else return __ldg(p);
}
// occupancy of cell (i, j) from the row-packed copy; outside the map = occupied
template <bool kS = false>
__device__ __forceinline__ bool occ_global(const MapDev& m, int i, int j) {
    if ((unsigned)i >= (unsigned)m.H || (unsigned)j >= (unsigned)m.W) return true;
    uint32_t w = map_word<kS>(m.row + (size_t)(i + kLineGuard) * m.strideR + ((j + kCellShift) >> 5));
    return (w >> (j & 31)) & 1u;
}

}  // namespace fn

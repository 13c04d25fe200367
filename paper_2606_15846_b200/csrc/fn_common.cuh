// fn_common.cuh -- shared device-side structures and helpers of libflashnav (sm_100a).
// Layouts are described in DESIGN.md "Data layout in HBM".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fn {

constexpr int kMaxVerts = 64;
constexpr int kMaxAttempts = 256;
constexpr int kNCounters = 8;
enum Counter { kRays = 0, kWords = 1, kResets = 2, kResetFail = 3, kNonFinite = 4, kEnvSteps = 5 };

// Bit-packed map, two orientations.  A "line" is one row of the row-packed copy (bits run along
// columns) or one column of the column-packed copy (bits run along rows).  Each line is
//   [1 pad word][nw data words][1 pad word]   (32-bit words, bit b of word k = cell 32k + b, pads = 0)
// so that a 64-bit window starting at any data word can be read with two aligned 32-bit loads.
struct MapDev {
    const uint32_t* row;     // [H][strideR]
    const uint32_t* col;     // [W][strideC]
    int H, W;
    int nwR, nwC;            // data words per line: ceil(W/32), ceil(H/32)
    int strideR, strideC;    // nw + 2
    float rho;               // metres per cell
    double inv_rho;          // 1 / (double)rho
};

// Per-env sensing pose, written by the env/reset kernels, read by the beam kernel.
struct __align__(32) PoseD {
    double ox, oy;           // sensor origin in cell units
    double c, s;             // cos/sin of the heading
};

struct RobotDev {
    const double2* beam_cs;  // [B] (cos, sin) of theta_j + s_psi
    const double2* verts;    // [V] footprint vertices, body frame, metres
    int B, V;
    int drive;               // 0 diff, 1 omni
    int A;                   // action dim
    float lim[6];
    float rmax;              // metres
    double T;                // rmax / rho in cells
    double sx, sy;           // sensor offset, metres
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
    double r = a - two_pi * floor((a + pi) / two_pi);
    if (r >= pi) r -= two_pi;
    if (r < -pi) r += two_pi;
    return r;
}

// occupancy of cell (i, j) from the row-packed copy in global memory; outside the map = occupied
__device__ __forceinline__ bool occ_global(const MapDev& m, int i, int j) {
    if ((unsigned)i >= (unsigned)m.H || (unsigned)j >= (unsigned)m.W) return true;
    uint32_t w = __ldg(m.row + (size_t)i * m.strideR + 1 + (j >> 5));
    return (w >> (j & 31)) & 1u;
}

}  // namespace fn

// fn_features.cuh -- clearance features: Eq. (3) of the paper and the sector
// min-pooling that turns the raw ranges into the policy's obstacle features z_t.
//
// Operation: each VALID range endpoint (range < r_max) is expressed in the body
// frame using the sensor placement, e_j = s_xy + r_j (cos, sin)(theta_j + s_psi); its distance to the
// footprint polygon is delta_j = min over the boundary segments (0 for points inside), capped at r_max;
// beams without a valid hit get r_max; z_k = min of delta_j over the beams of sector k.  Sector of beam j
// = floor(j n_sectors / B): n_sectors groups of consecutive beams in table order (reading G21).
//
// kFeatSplit warps per env: their lanes stride over the env's beams (coalesced reads of the range row, L2-resident
// right after the beam kernel), each computes its delta in fp32 (ample: the tolerance is 1e-4 m, delta is
// continuous across the polygon boundary) and the sector minima are kept in shared memory with atomicMin
// on the float bits (monotone for non-negative floats).
#pragma once
#include "fn_common.cuh"

namespace fn {

struct FeatArgs {
    const double2* beam_cs;      // [B] (cos, sin) of theta_j + s_psi
    const double2* verts;        // [V] footprint vertices, body frame, metres
    const int* nxt;              // [V] next vertex within the vertex's component (union of polygons)
    int B, V, n_sectors;
    float rmax, sx, sy;
    const float* ranges;         // [N][B]
    float* z;                    // [N][n_sectors]
    const int* list;             // compacted env indices or NULL (= all envs)
    const int* count_dev;        // number of listed envs (device) or NULL
    const int* list_par_dev;     // or NULL; else list += (*list_par_dev ^ 1) * n_all, count_dev += (*list_par_dev ^ 1)
    int n_all;
};

constexpr int kFeatWarps = 8;
constexpr int kFeatSplit = 4;                         // warps that share one env's beams (latency: an env's row is short)
constexpr int kFeatEnvs = kFeatWarps / kFeatSplit;   // envs a CTA works on at a time

__host__ __device__ inline size_t feat_smem_bytes(int V, int n_sectors) {
    return (size_t)V * 8 * sizeof(float) + (size_t)kFeatEnvs * n_sectors * sizeof(unsigned);
}
__host__ __device__ inline size_t feat_smem_bytes(int V, int n_sectors, int B) {
    return feat_smem_bytes(V, n_sectors) + (size_t)B * sizeof(float2);
}

__global__ void __launch_bounds__(kFeatWarps * 32) features_kernel(FeatArgs a) {
    extern __shared__ __align__(16) uint8_t s_dyn[];
    // beam directions as floats, then per edge k (vertex k -> nxt[k]): start a, direction e, 1/|e|^2, e_x/e_y,
    // end vertex y (the SAME float the edge from that vertex starts at, so the even-odd rule is consistent
    // at vertices) and whether the edge closes its component ("For a union of polygons, the minimum
    // distance over its components is used": inside = inside ANY component)
    // (two 16-byte records per edge, so the per-edge loop below issues two shared loads instead of eight)
    float4* s_e0 = reinterpret_cast<float4*>(s_dyn);               // start a (x, y), direction e (x, y)
    float4* s_e1 = s_e0 + a.V;                                     // 1/|e|^2, e_x/e_y, end vertex y, closes its component
    float2* s_cs = reinterpret_cast<float2*>(s_e1 + a.V);
    const int wib = threadIdx.x >> 5, grp = wib / kFeatSplit, sub = wib % kFeatSplit;   // env slot, warp within the env
    unsigned* s_z = reinterpret_cast<unsigned*>(s_cs + a.B) + grp * a.n_sectors;
    for (int j = threadIdx.x; j < a.B; j += blockDim.x) { const double2 c = a.beam_cs[j]; s_cs[j] = make_float2((float)c.x, (float)c.y); }
    for (int k = threadIdx.x; k < a.V; k += blockDim.x) {
        const int k1 = a.nxt[k];
        const double2 p = a.verts[k], q = a.verts[k1];
        const float ex = (float)(q.x - p.x), ey = (float)(q.y - p.y), l2 = ex * ex + ey * ey;
        s_e0[k] = make_float4((float)p.x, (float)p.y, ex, ey);
        s_e1[k] = make_float4(l2 > 0.0f ? 1.0f / l2 : 0.0f, ey != 0.0f ? ex / ey : 0.0f, (float)q.y, k1 <= k ? 1.0f : 0.0f);
    }
    __syncthreads();
    griddep_wait();                                                // the ranges come from the beam kernel
    griddep_launch_dependents();
    if (a.list_par_dev) { const int q = *a.list_par_dev ^ 1; a.list += (size_t)q * a.n_all; a.count_dev += q; }
    const int n_env = a.count_dev ? *a.count_dev : a.n_all;
    const int lane = threadIdx.x & 31;
    const unsigned rmax_bits = __float_as_uint(a.rmax);
    const unsigned long long invB = ~0ull / (unsigned long long)a.B + 1ull;          // floor(2^64 / B) + 1
    const int tid = sub * 32 + lane;                               // thread index within the env's group
    for (int le0 = blockIdx.x * kFeatEnvs; le0 < n_env; le0 += gridDim.x * kFeatEnvs) {       // (uniform over the CTA)
        const int le = le0 + grp;
        const bool have = le < n_env;
        const int e = have ? (a.list ? a.list[le] : le) : 0;
        for (int k = tid; k < a.n_sectors; k += kFeatSplit * 32) s_z[k] = rmax_bits;
        __syncthreads();
        const float* row = a.ranges + (size_t)e * a.B;
        if (have)
        for (int j0 = tid; j0 < a.B; j0 += 4 * kFeatSplit * 32) {  // four chunks per trip: their loads overlap
            float r[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) r[u] = j0 + kFeatSplit * 32 * u < a.B ? row[j0 + kFeatSplit * 32 * u] : a.rmax;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int j = j0 + kFeatSplit * 32 * u;
                if (j >= a.B) break;
                float d = a.rmax;                                  // no valid hit: the maximum range
                if (r[u] < a.rmax) {
                    const float2 cs = s_cs[j];
                    const float px = fmaf(r[u], cs.x, a.sx), py = fmaf(r[u], cs.y, a.sy);
                    float d2 = INFINITY;
                    bool inside = false, inside_c = false;
#pragma unroll 4
                    for (int k = 0; k < a.V; ++k) {
                        const float4 g0 = s_e0[k], g1 = s_e1[k];
                        const float ax = g0.x, ay = g0.y, ex = g0.z, ey = g0.w;
                        const float rx = px - ax, ry = py - ay;
                        const float t = fminf(fmaxf((rx * ex + ry * ey) * g1.x, 0.0f), 1.0f);
                        const float qx = rx - t * ex, qy = ry - t * ey;
                        d2 = fminf(d2, qx * qx + qy * qy);
                        if ((ay > py) != (g1.z > py) && rx < ry * g1.y) inside_c = !inside_c;       // even-odd rule
                        if (g1.w != 0.0f) { inside |= inside_c; inside_c = false; }
                    }
                    d = inside ? 0.0f : fminf(sqrtf(d2), a.rmax);  // capped at the sensor range
                }
                const unsigned k = a.B > 1 ? (unsigned)__umul64hi((unsigned long long)j * (unsigned)a.n_sectors, invB) : 0u;   // (B = 1: one sector)
                atomicMin(&s_z[k], __float_as_uint(d));
            }
        }
        __syncthreads();
        if (have) for (int k = tid; k < a.n_sectors; k += kFeatSplit * 32) a.z[(size_t)e * a.n_sectors + k] = __uint_as_float(s_z[k]);
        __syncthreads();
    }
}

}  // namespace fn

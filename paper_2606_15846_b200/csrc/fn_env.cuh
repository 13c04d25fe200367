// fn_env.cuh -- per-environment kernels: S1 clip + motion, S3 footprint collision, S4 goal obs /
// reward / done, S5 reset, S6 compaction of the reset mask.  One warp per environment.
// fp64 throughout for the geometry (per-env work is ~0.1 % of the beam work; B200 runs fp64 at half
// rate), so every decision sits far inside the 1e-5 cell near-tie margin of the parity contract.
#pragma once
#include "fn_common.cuh"

namespace fn {

// ---------------------------------------------------------------- S3: footprint collision
// Closed polygon vs closed occupied cell (the zero-sampling-interval limit of Eq. (2),
// PAPER.md:118-123): a cell collides iff some polygon edge meets its closed square, or the
// square's centre lies inside the polygon.  Edge vs square by the separating-axis test
// (axes x, y and the edge normal), centre by the even-odd crossing rule -- no divisions.
__device__ __forceinline__ bool cell_meets_polygon(int V, const double* vx, const double* vy, int j, int i) {
    const double xl = (double)j, xh = xl + 1.0, yl = (double)i, yh = yl + 1.0;
    const double cx = xl + 0.5, cy = yl + 0.5;
    bool inside = false;
    double px = vx[V - 1], py = vy[V - 1];
    for (int a = 0; a < V; ++a) {
        const double qx = vx[a], qy = vy[a];
        if (!(fmax(px, qx) < xl || fmin(px, qx) > xh || fmax(py, qy) < yl || fmin(py, qy) > yh)) {
            const double ex = qx - px, ey = qy - py;
            const double a0 = ex * (yl - py), a1 = ex * (yh - py);
            const double b0 = ey * (xl - px), b1 = ey * (xh - px);
            const double f00 = a0 - b0, f10 = a0 - b1, f01 = a1 - b0, f11 = a1 - b1;
            const double mn = fmin(fmin(f00, f10), fmin(f01, f11));
            const double mxv = fmax(fmax(f00, f10), fmax(f01, f11));
            if (mn <= 0.0 && mxv >= 0.0) return true;
        }
        if ((qy > cy) != (py > cy)) {
            const double ey = py - qy;
            const double t = (px - qx) * (cy - qy) - (cx - qx) * ey;   // sign(ey) * (x_cross - cx)
            if (ey > 0.0 ? t > 0.0 : t < 0.0) inside = !inside;
        }
        px = qx; py = qy;
    }
    return inside;
}

// Warp-cooperative: all lanes pass the same pose; svx/svy are this warp's shared scratch [kMaxVerts].
// Lanes transform the vertices, reduce the bounding window, then stride over its cells; only
// occupied (or outside-map) cells pay for the polygon test.  Returns the same flag on every lane.
__device__ bool warp_collision(const MapDev& m, const RobotDev& rb, double x, double y, double c,
                               double s, double* svx, double* svy) {
    const int lane = lane_id();
    const double rho = (double)m.rho;
    double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    __syncwarp();
    for (int k = lane; k < rb.V; k += 32) {
        const double2 f = rb.verts[k];
        const double wx = (x + c * f.x - s * f.y) / rho, wy = (y + s * f.x + c * f.y) / rho;
        svx[k] = wx; svy[k] = wy;
        xmin = fmin(xmin, wx); xmax = fmax(xmax, wx);
        ymin = fmin(ymin, wy); ymax = fmax(ymax, wy);
    }
    xmin = warp_min(xmin); xmax = warp_max(xmax); ymin = warp_min(ymin); ymax = warp_max(ymax);
    __syncwarp();
    if (!(isfinite(xmin) && isfinite(xmax) && isfinite(ymin) && isfinite(ymax))) return true;
    // a footprint reaching outside the map collides with the (occupied) outside at once
    if (xmin < 0.0 || ymin < 0.0 || xmax >= (double)m.W || ymax >= (double)m.H) return true;
    const int j0 = __double2int_rd(xmin), j1 = __double2int_rd(xmax);
    const int i0 = __double2int_rd(ymin), i1 = __double2int_rd(ymax);
    const int ncols = j1 - j0 + 1, total = ncols * (i1 - i0 + 1);
    bool found = false;
    for (int base = 0; base < total; base += 32) {
        const int n = base + lane;
        if (n < total) {
            const int i = i0 + n / ncols, j = j0 + n % ncols;
            if (occ_global(m, i, j)) found = cell_meets_polygon(rb.V, svx, svy, j, i);
        }
        if (__any_sync(0xffffffffu, found)) return true;
    }
    return false;
}

// ---------------------------------------------------------------- S1 + S3 + S4: the env step
struct EnvArgs {
    MapDev map;
    RobotDev robot;
    TaskDev task;
    int n;
    float dt;
    float* states;               // [8][n]
    const float* actions;        // [n][A]
    uint8_t* reset_mask;         // in: forced, out: done
    uint8_t* out_collision;
    float* out_goal_obs;         // [2][n]
    float* out_reward;           // or NULL
    float* d_prev;
    int* ep_step;
    PoseD* poses;
    int* pose_inside;
    float* ring;                 // or NULL
    unsigned long long ring_cap, ring_head;
    int ring_row;
    unsigned long long* counters;
};

__device__ __forceinline__ void write_pose(const MapDev& m, const RobotDev& rb, PoseD* out, int* inside,
                                           float xf, float yf, double c, double s) {
    const double rho = (double)m.rho;
    PoseD p;
    p.ox = ((double)xf + c * rb.sx - s * rb.sy) / rho;
    p.oy = ((double)yf + s * rb.sx + c * rb.sy) / rho;
    p.c = c; p.s = s;
    *out = p;
    // beams from here cannot leave the map: the beam kernel then skips its exit clipping
    const double lo = rb.T + 1.0;
    *inside = (p.ox >= lo && p.ox < (double)m.W - lo && p.oy >= lo && p.oy < (double)m.H - lo) ? 1 : 0;
}

__global__ void __launch_bounds__(256) env_step_kernel(EnvArgs a) {
    __shared__ double s_vx[8][kMaxVerts], s_vy[8][kMaxVerts];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = blockIdx.x * 8 + wib;
    if (e >= a.n) return;
    const int n = a.n;
    // ---- S1: clip ("within the configured bounds") and exact constant-twist step
    const double x = a.states[0 * n + e], y = a.states[1 * n + e], psi = a.states[2 * n + e];
    const float gxf = a.states[6 * n + e], gyf = a.states[7 * n + e];
    const int A = a.robot.A;
    float avx = a.actions[(size_t)e * A], avy = 0.0f, aw;
    if (a.robot.drive == 0) aw = a.actions[(size_t)e * A + 1];
    else { avy = a.actions[(size_t)e * A + 1]; aw = a.actions[(size_t)e * A + 2]; }
    const bool bad = !(isfinite(avx) && isfinite(avy) && isfinite(aw));
    avx = fminf(fmaxf(avx, a.robot.lim[0]), a.robot.lim[1]);
    if (a.robot.drive != 0) avy = fminf(fmaxf(avy, a.robot.lim[2]), a.robot.lim[3]);
    aw = fminf(fmaxf(aw, a.robot.lim[4]), a.robot.lim[5]);
    const double dt = (double)a.dt, vx = avx, vy = avy, w = aw;
    const double th = w * dt;
    double Ac, Cc;
    if (fabs(th) < 1e-8) { Ac = 1.0 - th * th / 6.0; Cc = 0.5 * th; }
    else { const double sh = sin(0.5 * th); Ac = sin(th) / th; Cc = sh * sh / (0.5 * th); }
    const double bx = dt * (Ac * vx - Cc * vy), by = dt * (Cc * vx + Ac * vy);
    double s0, c0;
    sincos(psi, &s0, &c0);
    const float xf = (float)(x + c0 * bx - s0 * by);
    const float yf = (float)(y + s0 * bx + c0 * by);
    const float psif = (float)wrap_pi(psi + th);
    // ---- sensing/collision pose = the stored fp32 pose, widened (parity is per step on stored bits)
    double s1, c1;
    sincos((double)psif, &s1, &c1);
    // ---- S3
    const bool col = warp_collision(a.map, a.robot, (double)xf, (double)yf, c1, s1, s_vx[wib], s_vy[wib]);
    // ---- S4: goal obs, reward Eq. (1), done
    const double gdx = (double)gxf - (double)xf, gdy = (double)gyf - (double)yf;
    const float d = (float)sqrt(gdx * gdx + gdy * gdy);
    const float alpha = (float)wrap_pi(atan2(gdy, gdx) - (double)psif);
    if (lane == 0) {
        const float dp = a.d_prev[e];
        const int es = a.ep_step[e];
        const bool reached = d < a.task.goal_tol;
        const float r = col ? a.task.r_collision
                            : reached ? a.task.r_success
                                      : (float)((double)a.task.c_progress * ((double)dp - (double)d));
        const bool limit = a.task.max_episode_steps > 0 && es + 1 >= a.task.max_episode_steps;
        const bool forced = a.reset_mask[e] != 0;
        const uint8_t done = (col || reached || limit || forced) ? 1 : 0;
        a.states[0 * n + e] = xf; a.states[1 * n + e] = yf; a.states[2 * n + e] = psif;
        a.states[3 * n + e] = avx; a.states[4 * n + e] = avy; a.states[5 * n + e] = aw;
        a.out_collision[e] = col ? 1 : 0;
        a.out_goal_obs[e] = d; a.out_goal_obs[n + e] = alpha;
        if (a.out_reward) a.out_reward[e] = r;
        a.reset_mask[e] = done;
        a.d_prev[e] = d;
        a.ep_step[e] = es + 1;
        write_pose(a.map, a.robot, &a.poses[e], &a.pose_inside[e], xf, yf, c1, s1);
        if (a.ring) {
            // complete this step's row (its obs part was written when that observation was produced)
            const int B = a.robot.B;
            float* row = a.ring + ((a.ring_head + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
            for (int k = 0; k < A; ++k) row[B + 5 + k] = a.actions[(size_t)e * A + k];
            row[B + 5 + A] = r;
            row[B + 6 + A] = done ? 1.0f : 0.0f;
            // and start the next step's row with the new goal obs and velocities
            float* nxt = a.ring + ((a.ring_head + (unsigned long long)n + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
            nxt[B] = d; nxt[B + 1] = alpha; nxt[B + 2] = avx; nxt[B + 3] = avy; nxt[B + 4] = aw;
        }
        if (bad) atomicAdd(&a.counters[kNonFinite], 1ull);
    }
}

// ---------------------------------------------------------------- S6: ordered compaction of a u8 mask
// One CTA of 1024 threads: thread t owns a contiguous segment, block-wide exclusive scan of the
// segment counts, then each thread writes its indices.  list is ascending; *count = number set.
__global__ void __launch_bounds__(1024) compact_mask_kernel(const uint8_t* mask, int n, int* list, int* count) {
    __shared__ int s_warp[32];
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    const int seg = (n + 1023) / 1024;
    const int lo = min(n, t * seg), hi = min(n, lo + seg);
    int c = 0;
    for (int i = lo; i < hi; ++i) c += mask[i] != 0;
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int v = s_warp[lane], iv = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, iv, o); if (lane >= o) iv += u; }
        s_warp[lane] = iv - v;
        if (lane == 31) *count = iv;
    }
    __syncthreads();
    int pos = s_warp[wid] + incl - c;
    for (int i = lo; i < hi; ++i) if (mask[i] != 0) list[pos++] = i;
}

// ---------------------------------------------------------------- S5: reset of the listed envs
// Reading G16: counter-based SplitMix64 draws, first accepted attempt in attempt order.
__device__ __forceinline__ unsigned long long splitmix64_at(unsigned long long sigma, unsigned long long c) {
    unsigned long long z = sigma + (c + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ float u24_at(unsigned long long sigma, unsigned long long c) {
    return __fmul_rn((float)(splitmix64_at(sigma, c) >> 40), 5.9604644775390625e-08f);
}

struct ResetArgs {
    MapDev map;
    RobotDev robot;
    TaskDev task;
    RegionsDev regions;
    int n;
    float* states;
    const int* list;
    const int* count_dev;
    const unsigned long long* seeds;
    float* out_goal_obs;
    float* d_prev;
    int* ep_step;
    PoseD* poses;
    int* pose_inside;
    float* ring;
    unsigned long long ring_cap, ring_head;
    int ring_row;
    unsigned long long* counters;
};

__global__ void __launch_bounds__(256) reset_kernel(ResetArgs a) {
    __shared__ double s_vx[8][kMaxVerts], s_vy[8][kMaxVerts];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int count = *a.count_dev;
    const int n = a.n;
    const double rho = (double)a.map.rho;
    const float two_pi_f = 6.28318530717958647692f, pi_f = 3.14159265358979323846f;
    const float dmin2 = __fmul_rn(a.task.dmin, a.task.dmin), dmax2 = __fmul_rn(a.task.dmax, a.task.dmax);
    for (int li = blockIdx.x * 8 + wib; li < count; li += gridDim.x * 8) {
        const int e = a.list[li];
        int r0 = 0, c0 = 0, rh = a.map.H, cw = a.map.W;
        if (a.regions.n > 0) { const int4 R = a.regions.rects[e % a.regions.n]; r0 = R.x; c0 = R.y; rh = R.z; cw = R.w; }
        const float X0 = (float)((double)c0 * rho), Xe = (float)((double)cw * rho);
        const float Y0 = (float)((double)r0 * rho), Ye = (float)((double)rh * rho);
        const unsigned long long sigma = a.seeds[e];
        float x = 0.f, y = 0.f, psi = 0.f;
        double sp = 0.0, cp = 1.0;
        bool ok = false;
        for (int k = 0; k < kMaxAttempts && !ok; ++k) {
            x = __fmaf_rn(u24_at(sigma, 3ull * k), Xe, X0);
            y = __fmaf_rn(u24_at(sigma, 3ull * k + 1ull), Ye, Y0);
            psi = __fmaf_rn(u24_at(sigma, 3ull * k + 2ull), two_pi_f, -pi_f);
            sincos((double)psi, &sp, &cp);
            ok = !warp_collision(a.map, a.robot, (double)x, (double)y, cp, sp, s_vx[wib], s_vy[wib]);
        }
        bool fail = !ok;
        float gx = x, gy = y;
        ok = false;
        for (int m = 0; m < kMaxAttempts && !ok; ++m) {
            const float ua = __fmaf_rn(2.0f, u24_at(sigma, 768ull + 2ull * m), -1.0f);
            const float ub = __fmaf_rn(2.0f, u24_at(sigma, 768ull + 2ull * m + 1ull), -1.0f);
            gx = __fmaf_rn(ua, a.task.dmax, x);
            gy = __fmaf_rn(ub, a.task.dmax, y);
            const float ddx = __fsub_rn(gx, x), ddy = __fsub_rn(gy, y);
            const float d2 = __fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy));
            if (!(d2 >= dmin2 && d2 <= dmax2)) continue;
            const int j = __double2int_rd((double)gx / rho), i = __double2int_rd((double)gy / rho);
            ok = i >= r0 && j >= c0 && i < r0 + rh && j < c0 + cw && !occ_global(a.map, i, j);
        }
        fail = fail || !ok;
        const double gdx = (double)gx - (double)x, gdy = (double)gy - (double)y;
        const float d = (float)sqrt(gdx * gdx + gdy * gdy);
        const float alpha = (float)wrap_pi(atan2(gdy, gdx) - (double)psi);
        if (lane == 0) {
            a.states[0 * n + e] = x; a.states[1 * n + e] = y; a.states[2 * n + e] = psi;
            a.states[3 * n + e] = 0.f; a.states[4 * n + e] = 0.f; a.states[5 * n + e] = 0.f;
            a.states[6 * n + e] = gx; a.states[7 * n + e] = gy;
            a.d_prev[e] = d;
            a.ep_step[e] = 0;
            if (a.out_goal_obs) { a.out_goal_obs[e] = d; a.out_goal_obs[n + e] = alpha; }
            write_pose(a.map, a.robot, &a.poses[e], &a.pose_inside[e], x, y, cp, sp);
            if (a.ring) {
                float* row = a.ring + ((a.ring_head + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
                const int B = a.robot.B;
                row[B] = d; row[B + 1] = alpha; row[B + 2] = 0.f; row[B + 3] = 0.f; row[B + 4] = 0.f;
            }
            atomicAdd(&a.counters[kResets], 1ull);
            if (fail) atomicAdd(&a.counters[kResetFail], 1ull);
        }
    }
}

// ---------------------------------------------------------------- observe-all support: poses from states
struct PoseArgs {
    MapDev map;
    RobotDev robot;
    int n;
    const float* states;
    float* out_goal_obs;         // or NULL
    PoseD* poses;
    int* pose_inside;
};
__global__ void __launch_bounds__(256) pose_from_state_kernel(PoseArgs a) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= a.n) return;
    const int n = a.n;
    const float x = a.states[e], y = a.states[n + e], psi = a.states[2 * n + e];
    double s, c;
    sincos((double)psi, &s, &c);
    write_pose(a.map, a.robot, &a.poses[e], &a.pose_inside[e], x, y, c, s);
    if (a.out_goal_obs) {
        const double gdx = (double)a.states[6 * n + e] - (double)x, gdy = (double)a.states[7 * n + e] - (double)y;
        a.out_goal_obs[e] = (float)sqrt(gdx * gdx + gdy * gdy);
        a.out_goal_obs[n + e] = (float)wrap_pi(atan2(gdy, gdx) - (double)psi);
    }
}

}  // namespace fn

// fn_env.cuh -- per-environment kernels: S1 clip + motion, S3 footprint collision, S4 goal obs /
// reward / done, S5 reset, S6 compaction of the reset mask.
// Geometry is fp64 (per-env work is ~1 % of the beam work; B200 runs fp64 at half rate), so every
// discrete decision sits ~10 orders of magnitude inside the 1e-5 cell near-tie margin of the parity
// contract.  The scalar math runs one THREAD per env (a warp-uniform fp64 instruction still occupies
// the fp64 pipe for the whole warp, so redundant lanes are not free); only the exact polygon test of
// the few envs whose footprint window holds occupied cells is warp-cooperative.
#pragma once
#include "fn_common.cuh"

namespace fn {

// ---------------------------------------------------------------- S3: footprint collision
// Closed polygon vs closed occupied cell = the zero-sampling-interval limit of Eq. (2)
// (PAPER.md:118-123); anything outside the map is occupied.
//
// Two stages.  (1) per thread: transform the vertices, take the bounding window of cells; a window
// that leaves the map collides at once; otherwise read the window's rows of occupancy bits -- no
// occupied cell in the window = no collision (the common case).  (2) warp-cooperative, only for
// windows holding occupied cells: one lane per window row builds the exact set of cells of that row
// that the closed polygon meets, as a bit mask, and ANDs it with the row's occupancy bits:
//   cells met by the polygon = cells some edge passes through  U  cells whose centre is inside
// (a cell no edge passes through lies wholly inside or wholly outside).  Per row, an edge clipped to
// the strip y in [i, i+1] covers the cells floor(x_a)..floor(x_b) of its x-extent; the centres inside
// follow from the even-odd rule on the line y = i + 1/2 (each crossing toggles the cells to its left).
// Cost: O(V) per row whatever the number of occupied cells.

struct Window {
    int i0, i1, j0, j1;      // inclusive cell ranges (rows, columns)
    int status;              // 0 = free (no occupied cell in the window), 1 = collides (leaves the map /
};                           //     non-finite), 2 = occupied cells in the window: exact test needed

// occupancy bits of row i, columns jb .. jb+31 (bit b = cell jb + b), from the row-packed copy
template <bool kS = false>
__device__ __forceinline__ uint32_t row_bits(const uint32_t* __restrict__ row, int strideR, int i, int jb) {
    const int q = jb + kCellShift;
    const uint32_t* p = row + (size_t)(i + kLineGuard) * strideR + (q >> 5);
    return __funnelshift_r(map_word<kS>(p), map_word<kS>(p + 1), q);
}
__device__ __forceinline__ uint32_t low_bits(int n) {           // n in [0, 32] -> n low bits set
    return n >= 32 ? 0xffffffffu : ((1u << n) - 1u);
}

// stage 1, one thread per pose.  verts = the footprint vertices (a shared-memory copy in the kernels).
// The window rows are read eight at a time so that their (independent, mostly L2-latency) loads overlap.
template <bool kS = false>
__device__ __forceinline__ Window footprint_window(const MapDev& m, const double2* __restrict__ verts, const int V,
                                                   double x, double y, double c, double s) {
    const double inv = m.inv_rho;
    double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    for (int k = 0; k < V; ++k) {
        const double2 f = verts[k];
        const double wx = (x + c * f.x - s * f.y) * inv, wy = (y + s * f.x + c * f.y) * inv;
        xmin = fmin(xmin, wx); xmax = fmax(xmax, wx);
        ymin = fmin(ymin, wy); ymax = fmax(ymax, wy);
    }
    Window w;
    w.i0 = w.i1 = w.j0 = w.j1 = 0;
    w.status = 1;
    // NaN-safe: a footprint reaching outside the map meets the (occupied) outside at once
    if (!(xmin >= 0.0 && ymin >= 0.0 && xmax < (double)m.W && ymax < (double)m.H)) return w;
    w.j0 = __double2int_rd(xmin); w.j1 = __double2int_rd(xmax);
    w.i0 = __double2int_rd(ymin); w.i1 = __double2int_rd(ymax);
    uint32_t any = 0;
    for (int jb = w.j0; jb <= w.j1; jb += 32) {
        const uint32_t cm = low_bits(w.j1 - jb + 1);
        for (int i = w.i0; i <= w.i1; i += 8) {
            uint32_t v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = row_bits<kS>(m.row, m.strideR, min(i + u, w.i1), jb);
#pragma unroll
            for (int u = 0; u < 8; ++u) any |= v[u];
        }
        any &= cm;
        if (any) break;
    }
    w.status = any ? 2 : 0;
    return w;
}

// stage 2, warp-cooperative over ALL of the warp's poses that need it at once: every such lane puts
// its transformed vertices and edge slopes into its slot of the warp's shared scratch, the window rows
// of all slots are numbered consecutively (prefix sum), and the lanes take these (slot, row) items 32
// at a time.  The cost is ceil(total rows / 32) passes of O(V) each instead of one pass per pose.
struct ColScratch {          // per warp, in dynamic shared memory
    double* vx;              // [32][V] vertex x (cells)
    double* vy;              // [32][V]
    double* sl;              // [32][V] edge k -> k+1: dx / dy
    int* pref;               // [32] first item of the slot (exclusive prefix sum of the row counts)
    int* win;                // [32][4] i0, j0, j1, -
    unsigned* hit;           // [1] bit per slot
    double2* verts;          // [V] copy of the footprint vertices (body frame, metres)
    int* nxt;                // [V] next vertex of each vertex within its component
};
__host__ __device__ inline size_t col_scratch_bytes(int V) { return (size_t)32 * 3 * V * 8 + (size_t)V * 16 + (size_t)((V + 3) / 4) * 16 + 32 * 4 + 32 * 16 + 16; }
__device__ __forceinline__ ColScratch col_scratch(uint8_t* base, int V) {
    ColScratch cs;
    cs.vx = reinterpret_cast<double*>(base);
    cs.vy = cs.vx + 32 * V;
    cs.sl = cs.vy + 32 * V;
    cs.verts = reinterpret_cast<double2*>(cs.sl + 32 * V);
    cs.pref = reinterpret_cast<int*>(cs.verts + V);
    cs.win = cs.pref + 32;
    cs.hit = reinterpret_cast<unsigned*>(cs.win + 32 * 4);
    cs.nxt = reinterpret_cast<int*>(cs.hit + 4);
    return cs;
}

// All 32 lanes must call; `need` = this lane's pose needs the exact test (window status 2).
// Returns true for a lane whose polygon meets an occupied cell (false for lanes that did not need it).
template <bool kS = false>
__device__ __noinline__ bool warp_collisions_exact(const uint32_t* __restrict__ row, const int strideR,
                                                   const double2* __restrict__ verts, const int* __restrict__ nxt, const int V,
                                                   const double inv, const bool need, const double x, const double y,
                                                   const double c, const double s, const int i0, const int i1,
                                                   const int j0, const int j1, const ColScratch cs) {
    const int lane = lane_id();
    __syncwarp();
    if (need) {
        double* vx = cs.vx + lane * V;
        double* vy = cs.vy + lane * V;
        double* sl = cs.sl + lane * V;
        for (int k = 0; k < V; ++k) {
            const double2 f = verts[k];
            vx[k] = (x + c * f.x - s * f.y) * inv;
            vy[k] = (y + s * f.x + c * f.y) * inv;
        }
        for (int k = 0; k < V; ++k) {                              // edge k: vertex k -> nxt[k] (within its component)
            const int k1 = nxt[k];
            const double dy = vy[k1] - vy[k];
            double r = 0.0;
            if (dy != 0.0) {                                       // 1 / dy: one Newton step on the 20-bit
                double r0;                                         // reciprocal (relative error ~2^-40)
                asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0) : "d"(dy));
                r = fma(fma(-dy, r0, 1.0), r0, r0);
            }
            sl[k] = (vx[k1] - vx[k]) * r;
        }
        cs.win[lane * 4 + 0] = i0; cs.win[lane * 4 + 1] = j0; cs.win[lane * 4 + 2] = j1;
    }
    const int rows = need ? i1 - i0 + 1 : 0;
    int incl = rows;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    cs.pref[lane] = incl - rows;
    if (lane == 0) *cs.hit = 0u;
    __syncwarp();
    for (int t0 = 0; t0 < total; t0 += 32) {
        const int t = t0 + lane;
        if (t < total) {
            int slot = 0;                                          // last slot whose first item is <= t
#pragma unroll
            for (int st = 16; st > 0; st >>= 1) if (cs.pref[slot + st] <= t) slot += st;
            const int i = cs.win[slot * 4] + (t - cs.pref[slot]);
            const int sj0 = cs.win[slot * 4 + 1], sj1 = cs.win[slot * 4 + 2];
            const double* vx = cs.vx + slot * V;
            const double* vy = cs.vy + slot * V;
            const double* sl = cs.sl + slot * V;
            const double ylo_s = (double)i, yhi_s = ylo_s + 1.0, yc = ylo_s + 0.5;
            bool found = false;
            for (int jb = sj0; jb <= sj1 && !found; jb += 32) {
                const uint32_t occ = row_bits<kS>(row, strideR, i, jb) & low_bits(sj1 - jb + 1);
                if (occ == 0u) continue;
                // a footprint may be a union of polygons: the edges of a component are
                // consecutive and close on themselves (nxt[k] <= k at its last vertex); the cells inside
                // the union are the OR of the components' even-odd masks
                uint32_t touch = 0, inside = 0, inside_c = 0;
                for (int k = 0; k < V; ++k) {                      // edge k: vertex k -> nxt[k]
                    const int k1 = nxt[k];
                    const double px = vx[k], py = vy[k], qx = vx[k1], qy = vy[k1], sk = sl[k];
                    const double elo = fmin(py, qy), ehi = fmax(py, qy);
                    if (ehi >= ylo_s && elo <= yhi_s) {            // the edge meets the closed strip
                        const double exlo = fmin(px, qx), exhi = fmax(px, qx);
                        double xa = exlo, xb = exhi;
                        if (py != qy) {
                            const double x1 = px + (fmax(elo, ylo_s) - py) * sk, x2 = px + (fmin(ehi, yhi_s) - py) * sk;
                            xa = fmax(fmin(x1, x2), exlo); xb = fmin(fmax(x1, x2), exhi);
                        }
                        const int ca = max(__double2int_rd(xa) - jb, 0), cb = min(__double2int_rd(xb) - jb, 31);
                        if (ca <= cb) touch |= low_bits(cb + 1) & ~low_bits(ca);
                    }
                    if ((py > yc) != (qy > yc)) {                   // crosses the centre line: cells with
                        const double xc = px + (yc - py) * sk;      // centre j + 1/2 < xc lie to its left
                        const int nleft = __double2int_ru(xc - 0.5) - jb;
                        inside_c ^= low_bits(min(max(nleft, 0), 32));
                    }
                    if (k1 <= k) { inside |= inside_c; inside_c = 0u; }
                }
                found = (occ & (touch | inside)) != 0u;
            }
            if (found) atomicOr(cs.hit, 1u << slot);
        }
    }
    __syncwarp();
    return need && ((*cs.hit >> lane) & 1u);
}

// Per-lane collision flag from the window status (all 32 lanes must call).
template <bool kS = false>
__device__ __forceinline__ bool resolve_collisions(const MapDev& m, const RobotDev& rb, const Window& w,
                                                   double x, double y, double c, double s, const ColScratch cs) {
    const bool need = w.status == 2;
    bool col = w.status == 1;
    if (__any_sync(0xffffffffu, need))
        col |= warp_collisions_exact<kS>(m.row, m.strideR, cs.verts, cs.nxt, rb.V, m.inv_rho, need, x, y, c, s,
                                     w.i0, w.i1, w.j0, w.j1, cs);
    return col;
}

// ---------------------------------------------------------------- sensing pose for the beam kernel
// BeamPose (fn_common.cuh): sensor origin in cells and, for both choices of the dominant axis, the
// origin's fixed-point coordinate, the offset to the first line boundary and the address of the
// origin's line.
template <bool kS = false>
__device__ __forceinline__ BeamPose make_pose(const MapDev& m, const RobotDev& rb,
                                              float xf, float yf, float psif, double c, double s, const int sensor = 0) {
    const double ox = ((double)xf + c * rb.sxs[sensor] - s * rb.sys[sensor]) * m.inv_rho;
    const double oy = ((double)yf + s * rb.sxs[sensor] + c * rb.sys[sensor]) * m.inv_rho;
    BeamPose p;
    p.c = c; p.s = s;
    p.psi_bits = __float_as_int(psif);
    const bool in = ox >= 0.0 && ox < (double)m.W && oy >= 0.0 && oy < (double)m.H;   // false for NaN
    const int jx = in ? __double2int_rd(ox) : 0, iy = in ? __double2int_rd(oy) : 0;
    p.state = !in ? 2 : (occ_global<kS>(m, iy, jx) ? 1 : 0);
    const double fx = ox - (double)jx, fy = oy - (double)iy;
    const unsigned rowBytes = (unsigned)(m.H + 2 * kLineGuard) * (unsigned)m.strideR * 4u;
    p.o[0].ouM = ox + ((double)kCellShift + kMagic); p.o[0].h = 0.5 - fy; p.o[0].cu0 = jx;
    p.o[0].line_off = (unsigned)(iy + kLineGuard) * (unsigned)m.strideR * 4u;
    p.o[1].ouM = oy + ((double)kCellShift + kMagic); p.o[1].h = 0.5 - fx; p.o[1].cu0 = iy;
    p.o[1].line_off = rowBytes + (unsigned)(jx + kLineGuard) * (unsigned)m.strideC * 4u;
    p.line_par[0] = (unsigned)(iy + kLineGuard) & 1u; p.line_par[1] = (unsigned)(jx + kLineGuard) & 1u;
    p.o[0].ouMS = p.o[0].ouM + (double)(p.o[0].line_off << 3);
    p.o[1].ouMS = p.o[1].ouM + (double)((p.o[1].line_off - rowBytes) << 3);
    return p;
}
// the poses of the other sensors of a robot with several (sensor 0's is stored by the caller): poses[k * n + e]
template <bool kS = false>
__device__ __forceinline__ void write_more_poses(const MapDev& m, const RobotDev& rb, BeamPose* poses, const int n, const int e,
                                                 float xf, float yf, float psif, double c, double s) {
    for (int k = 1; k < rb.n_sensors; ++k) poses[(size_t)k * n + e] = make_pose<kS>(m, rb, xf, yf, psif, c, s, k);
}
template <bool kS = false>
__device__ __forceinline__ void write_pose(const MapDev& m, const RobotDev& rb, BeamPose* poses, const int n, const int e,
                                           float xf, float yf, float psif, double c, double s) {
    poses[e] = make_pose<kS>(m, rb, xf, yf, psif, c, s);
    write_more_poses<kS>(m, rb, poses, n, e, xf, yf, psif, c, s);
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
    BeamPose* poses;
    float* ring;                 // or NULL
    unsigned long long ring_cap;
    const unsigned long long* ring_head_dev;   // device: slot of env 0's pending row
    int ring_row;
    int epw;                     // envs per warp (1..32): lanes >= epw idle in the scalar part
    unsigned* beam_task_counter; // zeroed here for the beam kernel that follows
    int* done_list;              // [2][n] envs that report done (any order), one list per step parity;
    int* done_count;             // [2]    fn_reset(mask = NULL) uses the step's list.  The parity lives on
    const int* par_dev;          // the device (flipped by the step's beam kernel, which also clears the other
                                 // count), so a captured sequence of steps replays for any length
    uint8_t* eval_outcome;       // evaluation mode or NULL: 0 running, 1 success, 2 collision,
    float* eval_return;          //   3 step limit, 4 inactive slot; completed cases are frozen
    int eval_limit;
    unsigned long long* counters;
};

// One warp per CTA, `epw` envs per warp.  The exact polygon tests of a warp's envs run one after the
// other (each warp-cooperative), so small batches use few envs per warp to spread that serial chain
// over many warps and SMs (the scalar part is latency-bound there anyway); large batches use all 32
// lanes for throughput.
constexpr int kEnvBlock = 32;

// ---------------------------------------------------------------- S1: the motion update of one env
// Pure function of the stored state, the action and the stored sensing pose (no writes): the new fp32 pose
// and applied velocities, and cos/sin of the new heading in fp64.  `el` = the env to read.
struct EnvMotion {
    float xf, yf, psif, avx, avy, aw;
    double c1, s1;
    bool bad;                    // a non-finite action component
};
__device__ __forceinline__ EnvMotion env_motion(const EnvArgs& a, const int el) {
    const int n = a.n;
    const int es = a.ep_step[el];
    const int A = a.robot.A;
    // ---- S1: clip ("within the configured bounds") and exact constant-twist step
    const double x = a.states[0 * n + el], y = a.states[1 * n + el], psi = a.states[2 * n + el];
    float avx = a.actions[(size_t)el * A], avy = 0.0f, aw;
    if (a.robot.drive == 0) aw = a.actions[(size_t)el * A + 1];
    else { avy = a.actions[(size_t)el * A + 1]; aw = a.actions[(size_t)el * A + 2]; }
    const bool bad = !(isfinite(avx) && isfinite(avy) && isfinite(aw));
    avx = fminf(fmaxf(avx, a.robot.lim[0]), a.robot.lim[1]);
    if (a.robot.drive != 0) avy = fminf(fmaxf(avy, a.robot.lim[2]), a.robot.lim[3]);
    aw = fminf(fmaxf(aw, a.robot.lim[4]), a.robot.lim[5]);
    // acceleration limits (reading G2): previous applied velocity +- a_max dt, single fused fp32 operations
    if (a.robot.acc[0] < INFINITY) {
        const float vp = a.states[3 * n + el];
        avx = fminf(fmaxf(avx, __fmaf_rn(-a.robot.acc[0], a.dt, vp)), __fmaf_rn(a.robot.acc[0], a.dt, vp));
    }
    if (a.robot.drive != 0 && a.robot.acc[1] < INFINITY) {
        const float vp = a.states[4 * n + el];
        avy = fminf(fmaxf(avy, __fmaf_rn(-a.robot.acc[1], a.dt, vp)), __fmaf_rn(a.robot.acc[1], a.dt, vp));
    }
    if (a.robot.acc[2] < INFINITY) {
        const float vp = a.states[5 * n + el];
        aw = fminf(fmaxf(aw, __fmaf_rn(-a.robot.acc[2], a.dt, vp)), __fmaf_rn(a.robot.acc[2], a.dt, vp));
    }
    const double dt = (double)a.dt, vx = avx, vy = avy, w = aw;
    const double th = w * dt;
    // one sincos (of theta / 2) gives the integrator's A = sin(theta)/theta, C = sin^2(theta/2)/(theta/2)
    // and the rotation by theta
    double sh, ch;
    sincos(0.5 * th, &sh, &ch);
    const double sin_th = 2.0 * sh * ch, cos_th = 1.0 - 2.0 * sh * sh;
    double Ac, Cc;
    if (fabs(th) < 1e-8) { Ac = 1.0 - th * th / 6.0; Cc = 0.5 * th; }
    else { const double inv = 1.0 / th; Ac = sin_th * inv; Cc = 2.0 * sh * sh * inv; }
    const double bx = dt * (Ac * vx - Cc * vy), by = dt * (Cc * vx + Ac * vy);
    // cos/sin of the stored heading: kept in the sensing pose by the kernel that wrote that heading
    // (recomputed if the caller changed the state plane behind the sim's back)
    const BeamPose* pp = a.poses + el;
    double s0 = pp->s, c0 = pp->c;
    const float psi_f = a.states[2 * n + el];
    const bool fresh = pp->psi_bits == __float_as_int(psi_f);
    if (!fresh) sincos(psi, &s0, &c0);
    const float xf = (float)(x + c0 * bx - s0 * by);
    const float yf = (float)(y + s0 * bx + c0 * by);
    const double pw = wrap_pi(psi + th);
    const float psif = (float)pw;
    // ---- sensing/collision pose = the stored fp32 pose, widened (parity is per step on stored bits):
    // rotate (c0, s0) by theta, then by the fp32 rounding of the new heading (second order; < 1e-20);
    // an exact sincos every 32nd step of an episode bounds the accumulated rounding (~2e-16 per step)
    double s1, c1;
    if (fresh && (es & 31) != 31) {
        const double cr = c0 * cos_th - s0 * sin_th, sr = s0 * cos_th + c0 * sin_th;
        const double dl = (double)psif - pw;
        c1 = cr - sr * dl - 0.5 * cr * dl * dl;
        s1 = sr + cr * dl - 0.5 * sr * dl * dl;
    } else {
        sincos((double)psif, &s1, &c1);
    }
    EnvMotion mo;
    mo.xf = xf; mo.yf = yf; mo.psif = psif; mo.avx = avx; mo.avy = avy; mo.aw = aw; mo.c1 = c1; mo.s1 = s1; mo.bad = bad;
    return mo;
}
// the motion's results written back: state planes 0-5 and the sensing pose (all lanes that are live)
template <bool kS>
__device__ __forceinline__ void env_motion_store(const EnvArgs& a, const MapDev& m, const int e, const EnvMotion& mo,
                                                 BeamPose* pose_copy = nullptr) {
    const int n = a.n;
    a.states[0 * n + e] = mo.xf; a.states[1 * n + e] = mo.yf; a.states[2 * n + e] = mo.psif;
    a.states[3 * n + e] = mo.avx; a.states[4 * n + e] = mo.avy; a.states[5 * n + e] = mo.aw;
    const BeamPose bp = make_pose<kS>(m, a.robot, mo.xf, mo.yf, mo.psif, mo.c1, mo.s1);
    a.poses[e] = bp;
    write_more_poses<kS>(m, a.robot, a.poses, n, e, mo.xf, mo.yf, mo.psif, mo.c1, mo.s1);
    if (pose_copy) *pose_copy = bp;
    if (mo.bad) atomicAdd(&a.counters[kNonFinite], 1ull);
}
// the same values read back from memory (split step: the motion ran in an earlier kernel)
__device__ __forceinline__ EnvMotion env_motion_load(const EnvArgs& a, const int el) {
    const int n = a.n;
    EnvMotion mo;
    mo.xf = a.states[0 * n + el]; mo.yf = a.states[1 * n + el]; mo.psif = a.states[2 * n + el];
    mo.avx = a.states[3 * n + el]; mo.avy = a.states[4 * n + el]; mo.aw = a.states[5 * n + el];
    mo.c1 = a.poses[el].c; mo.s1 = a.poses[el].s; mo.bad = false;
    return mo;
}

// ---------------------------------------------------------------- S3 + S4 of one env per lane
// Collision at the new pose, goal observation, reward, done, the done list, the ring row and the episode
// bookkeeping.  All 32 lanes of the warp call (the exact polygon test is warp-cooperative); lanes with
// in_range = false idle and write nothing.  m = the packed map to read: a.map (kS = false) or the same map
// with row / col pointing at a shared-memory copy (kS = true).  ring_head = slot of env 0's row of THIS step.
// store_motion: also write the motion's results (the single-kernel env step); false when an earlier kernel
// stored them (split step).
// Returns the ballot of the lanes whose env reports done.
template <bool kS>
__device__ __forceinline__ unsigned env_outcome(const EnvArgs& a, const MapDev& m, const ColScratch& scratch, const int e,
                                            const int el, const bool in_range, const int lane, const EnvMotion& mo,
                                            const unsigned long long ring_head, const bool store_motion) {
    const int n = a.n;
    const bool frozen = in_range && a.eval_outcome != nullptr && a.eval_outcome[el] != 0;
    const bool live = in_range && !frozen;
    const float xf = mo.xf, yf = mo.yf, psif = mo.psif, avx = mo.avx, avy = mo.avy, aw = mo.aw;
    const double c1 = mo.c1, s1 = mo.s1;
    const float gxf = a.states[6 * n + el], gyf = a.states[7 * n + el];
    const float dp = a.d_prev[el];
    const int es = a.ep_step[el];
    const bool forced = a.reset_mask[el] != 0;
    const int A = a.robot.A;
    // ---- S3
    Window win = footprint_window<kS>(m, scratch.verts, a.robot.V, (double)xf, (double)yf, c1, s1);
    if (!live) win.status = 0;
    const bool col = resolve_collisions<kS>(m, a.robot, win, (double)xf, (double)yf, c1, s1, scratch);
    // ---- S4: goal obs, reward Eq. (1), done
    const double gdx = (double)gxf - (double)xf, gdy = (double)gyf - (double)yf;
    const float d = (float)sqrt(gdx * gdx + gdy * gdy);
    const float alpha = (float)wrap_pi(atan2(gdy, gdx) - (double)psif);
    const bool reached = d < a.task.goal_tol;
    const float r = col ? a.task.r_collision
                        : reached ? a.task.r_success
                                  : (float)((double)a.task.c_progress * ((double)dp - (double)d));
    const int step_limit = a.eval_outcome ? a.eval_limit : a.task.max_episode_steps;
    const bool limit = step_limit > 0 && es + 1 >= step_limit;
    const uint8_t done = (live && (col || reached || limit || forced)) ? 1 : 0;
    // the done envs, appended to the step's list (one atomic per warp): "Ended only" needs no mask scan
    const unsigned dm = __ballot_sync(0xffffffffu, done != 0);
    if (dm) {
        int base = 0;
        const int par = *a.par_dev;
        if (lane == 0) base = atomicAdd(a.done_count + par, __popc(dm));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (done) a.done_list[(size_t)par * n + base + __popc(dm & ((1u << lane) - 1u))] = e;
    }
    if (frozen) {                                                  // no state change, no reward, not done again
        a.reset_mask[e] = 0;
        if (a.out_reward) a.out_reward[e] = 0.0f;
    }
    if (!live) return dm;
    if (a.eval_outcome) {                                          // each case is recorded once
        a.eval_return[e] += r;
        if (done) a.eval_outcome[e] = col ? 2 : reached ? 1 : 3;
    }
    if (store_motion) env_motion_store<kS>(a, m, e, mo);
    a.out_collision[e] = col ? 1 : 0;
    a.out_goal_obs[e] = d; a.out_goal_obs[n + e] = alpha;
    if (a.out_reward) a.out_reward[e] = r;
    a.reset_mask[e] = done;
    a.d_prev[e] = d;
    a.ep_step[e] = es + 1;
    if (a.ring) {
        // complete this step's row (its obs part was written when that observation was produced)
        const int B = a.robot.B;
        const unsigned long long head = ring_head;
        float* row = a.ring + ((head + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
        for (int k = 0; k < A; ++k) row[B + 5 + k] = a.actions[(size_t)e * A + k];   // the raw action
        row[B + 5 + A] = r;
        row[B + 6 + A] = done ? ((col || reached) ? 1.0f : 2.0f) : 0.0f;   // 1 terminated, 2 truncated (limit / forced)
        // and start the next step's row with the new goal obs and velocities
        float* nxt = a.ring + ((head + (unsigned long long)n + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
        nxt[B] = d; nxt[B + 1] = alpha; nxt[B + 2] = avx; nxt[B + 3] = avy; nxt[B + 4] = aw;
    }
    return dm;
}

__global__ void __launch_bounds__(kEnvBlock) env_step_kernel(EnvArgs a) {
    extern __shared__ __align__(16) uint8_t s_dyn[];
    const ColScratch scratch = col_scratch(s_dyn, a.robot.V);
    for (int k = threadIdx.x; k < a.robot.V; k += kEnvBlock) { scratch.verts[k] = a.robot.verts[k]; scratch.nxt[k] = a.robot.nxt[k]; }
    __syncwarp();
    griddep_wait();                                                // states / actions / mask come from earlier work
    griddep_launch_dependents();                                   // the beam kernel may start staging the map now
    if (blockIdx.x == 0 && threadIdx.x == 0) *a.beam_task_counter = 0u;
    const int e = blockIdx.x * a.epw + threadIdx.x;
    const int n = a.n;
    const bool in_range = (int)threadIdx.x < a.epw && e < n;
    const int el = in_range ? e : n - 1;                           // idle lanes shadow the last env, write nothing
    const EnvMotion mo = env_motion(a, el);
    env_outcome<false>(a, a.map, scratch, e, el, in_range, (int)threadIdx.x, mo, a.ring ? *a.ring_head_dev : 0ull, true);
}

// advances the replay ring's head by n rows (one thread), after the env-step kernel of fn_step;
// head[1] counts the rows completed so far (the sampler's `filled` = min(head[1], capacity))
__global__ void ring_advance_kernel(unsigned long long* head, unsigned long long n, unsigned long long cap) {
    griddep_wait();
    griddep_launch_dependents();
    head[0] = (head[0] + n) % cap;
    head[1] += n;
    head[3] = head[2];                                             // terminal observations: a new batch starts (TerminalDev)
}

// ---------------------------------------------------------------- NEXT-2: uniform replay sampling
// "Each replay batch contains U x B transitions sampled uniformly from replay".  Sample i =
// the ring row at slot floor(SplitMix64(seed, i) filled / 2^64) (reading G22); optionally the next
// observation = the obs part of the same env's next row (slot + n_envs mod capacity).  A gather of
// whole rows: one warp per sample, lanes stride over the row (rows start at 4-byte alignment only), so
// every warp instruction moves 128 contiguous bytes; the kernel is HBM-bound.
__device__ __forceinline__ unsigned long long splitmix64_at(unsigned long long sigma, unsigned long long c);
// Terminal observations ("Observations before reset are retained as next observations in replay"): a
// second ring of t_cap entries of [ranges(B), d, alpha, v_x, v_y, w]; idx[ring slot] = the entry of that row,
// id[entry] = the global id of the row the entry belongs to, start[entry] = the entries written when the step the
// row belongs to ended.  The entries written by the resets after one step form a batch, given up as a whole as soon
// as a later write reuses one of them: an entry is kept while its id matches and head[0] <= start + t_cap (so what
// is kept does not depend on the order in which the envs of a reset are taken).
struct TerminalDev {
    float* term;                         // [t_cap][obs] or NULL = none attached
    int* idx;                            // [ring capacity], -1 = none
    unsigned long long* id;              // [t_cap]
    unsigned long long* start;           // [t_cap]
    unsigned long long* head;            // [2]: entries ever written; its value when the last step ended (= ring head words 2, 3)
    unsigned long long t_cap;
};
__device__ __forceinline__ bool terminal_kept(const TerminalDev& td, const unsigned long long slot, const unsigned long long g,
                                              const unsigned long long head_now) {
    const int t = td.idx[slot];
    return t >= 0 && td.id[t] == g && head_now <= td.start[t] + td.t_cap;
}
struct SampleArgs {
    const float* ring;
    const unsigned long long* head;      // [2]: head, rows completed
    unsigned long long cap, seed;
    int n_envs, row, obs, n_samples;
    float* out_rows;                     // [n_samples][row]
    float* out_next_obs;                 // [n_samples][obs] or NULL
    TerminalDev td;
};
__global__ void __launch_bounds__(256) ring_sample_kernel(SampleArgs a) {
    griddep_wait();
    griddep_launch_dependents();
    // completed rows outside the pending window [head, head + n_envs): the oldest at head - valid (reading G22)
    const unsigned long long total = a.head[1], head = a.head[0];
    const unsigned long long room = a.cap - (unsigned long long)a.n_envs;          // (cap >= 2 n_envs: fn_ring_attach)
    const unsigned long long valid = total < room ? total : room;
    if (valid == 0ull) return;
    const unsigned long long first = head + a.cap - valid;
    const int lane = threadIdx.x & 31;
    for (int i = blockIdx.x * 8 + (threadIdx.x >> 5); i < a.n_samples; i += gridDim.x * 8) {
        const unsigned long long si = __umul64hi(splitmix64_at(a.seed, (unsigned long long)i), valid);
        unsigned long long slot = first + si;
        if (slot >= a.cap) slot -= a.cap;
        if (slot >= a.cap) slot -= a.cap;
        const unsigned long long g = total - valid + si;           // global id of the sampled row
        const float* src = a.ring + slot * (unsigned long long)a.row;
        float* dst = a.out_rows + (size_t)i * a.row;
        // done code of the sampled copy: a truncated row (2) whose pre-reset observation is not kept becomes 3
        const float code = __ldg(src + a.row - 1);
        const float* nsrc = a.ring + ((slot + (unsigned long long)a.n_envs) % a.cap) * (unsigned long long)a.row;
        float code_out = code;
        if (code != 0.0f) {
            bool kept = false;
            if (a.td.term && terminal_kept(a.td, slot, g, a.td.head[0])) {
                nsrc = a.td.term + (unsigned long long)a.td.idx[slot] * (unsigned long long)a.obs;
                kept = true;
            }
            if (code == 2.0f && !kept) code_out = 3.0f;
        }
        for (int k = lane; k < a.row; k += 32) dst[k] = k == a.row - 1 ? code_out : __ldg(src + k);
        if (a.out_next_obs) {
            float* ndst = a.out_next_obs + (size_t)i * a.obs;
            for (int k = lane; k < a.obs; k += 32) ndst[k] = __ldg(nsrc + k);
        }
    }
}

// Before a reset overwrites them: the observation the last step left in the pending rows of the listed envs goes
// into the terminal ring, for every env whose last completed row (slot head - n + e, id total - n + e) has a done
// code != 0 and is not kept yet.  One warp per listed env; entries are taken with one atomic per env (any order: a
// call takes the same range of entries whatever the order, so what an old entry loses does not depend on it).
struct TerminalSaveArgs {
    const float* ring;
    const unsigned long long* head;      // [2]: head, rows completed
    unsigned long long cap;
    int n_envs, row, obs;
    const int* list;
    const int* count_dev;
    const int* list_par_dev;             // or NULL (see ResetArgs)
    TerminalDev td;
};
__global__ void __launch_bounds__(256) terminal_save_kernel(TerminalSaveArgs a) {
    griddep_wait();
    griddep_launch_dependents();
    const unsigned long long total = a.head[1], head = a.head[0];
    if (total < (unsigned long long)a.n_envs) return;              // no step has completed a row yet
    const int* list = a.list;
    const int* count_dev = a.count_dev;
    if (a.list_par_dev) { const int q = *a.list_par_dev ^ 1; list += (size_t)q * a.n_envs; count_dev += q; }
    const int count = *count_dev;
    const int lane = threadIdx.x & 31;
    const unsigned long long batch_start = a.td.head[1];
    for (int k = blockIdx.x * 8 + (threadIdx.x >> 5); k < count; k += gridDim.x * 8) {
        const unsigned long long e = (unsigned long long)list[k];
        const unsigned long long c = (head + a.cap - (unsigned long long)a.n_envs + e) % a.cap;
        const unsigned long long g = total - (unsigned long long)a.n_envs + e;
        if (a.ring[c * (unsigned long long)a.row + (unsigned long long)(a.row - 1)] == 0.0f) continue;
        // kept already (a reset called twice)?  Such an entry belongs to this batch, and a batch has at most n <= t_cap
        // entries, so whatever this launch has added meanwhile, head[0] <= start + t_cap holds for it.
        if (terminal_kept(a.td, c, g, a.td.head[0])) continue;
        unsigned long long entry = 0ull;
        if (lane == 0) entry = atomicAdd(a.td.head, 1ull) % a.td.t_cap;
        entry = __shfl_sync(0xffffffffu, entry, 0);
        const float* src = a.ring + ((head + e) % a.cap) * (unsigned long long)a.row;
        float* dst = a.td.term + entry * (unsigned long long)a.obs;
        int q = lane;
        for (; q + 224 < a.obs; q += 256) {                        // eight independent 128-byte loads in flight per warp
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = __ldg(src + q + 32 * u);
#pragma unroll
            for (int u = 0; u < 8; ++u) dst[q + 32 * u] = v[u];
        }
        for (; q < a.obs; q += 32) dst[q] = __ldg(src + q);
        if (lane == 0) { a.td.id[entry] = g; a.td.start[entry] = batch_start; a.td.idx[c] = (int)entry; }
    }
}

// ---------------------------------------------------------------- S6: ordered compaction of a u8 mask
// One CTA of 1024 threads: thread t owns a contiguous segment, block-wide exclusive scan of the
// segment counts, then each thread writes its indices.  list is ascending; *count = number set.
__global__ void __launch_bounds__(1024) compact_mask_kernel(const uint8_t* mask, int n, int* list, int* count) {
    __shared__ int s_warp[32];
    griddep_wait();
    griddep_launch_dependents();
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
// One warp per listed env; the 32 lanes evaluate 32 consecutive attempts at once and the first
// accepted one in ATTEMPT order wins (ballot + ffs), so the result equals the sequential rule.
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
    const int* list_par_dev;     // or NULL; else list += (*list_par_dev ^ 1) * n, count_dev += (*list_par_dev ^ 1)
    const unsigned long long* seeds;
    float* out_goal_obs;
    float* d_prev;
    int* ep_step;
    BeamPose* poses;
    float* ring;
    unsigned long long ring_cap;
    const unsigned long long* ring_head_dev;
    int ring_row;
    unsigned* beam_task_counter; // zeroed here for the beam kernel that follows
    unsigned long long* counters;
    uint8_t* fail_out;           // or NULL; else [n]: "no attempt was accepted" is stored here instead of counted
};

struct StepEnd {                         // device words owned by the sim, zero at creation
    unsigned done_ctas;                  // CTAs of the running launch that have finished
    unsigned outcomes_done;              // outcome warps of the running step that have finished (done list, prepared
                                         //   resets): zeroed by the step's motion kernel, read by prepared_reset_kernel
    int par_used;                        // the done-list parity that step fills
    unsigned pad_;
};

// A reset prepared ahead of fn_reset (fn_sim_prepare_reset): the step's outcome warps run reset_env for the envs
// they report done, with ResetArgs that point here instead of at the caller's arrays; fn_reset(mask = NULL) then
// only copies (reset_apply) and casts the beams.  Same layouts as the arrays they stand for.
struct PreparedReset {
    float* states;               // [8][n], NULL = nothing prepared
    float* goal_obs;             // [2][n]
    float* d_prev;               // [n]
    BeamPose* poses;             // [n]
    uint8_t* fail;               // [n]
};

constexpr int kResetWarps = 4;

// Reset of env e by one warp (all 32 lanes call).  m = the packed map to read: a.map (kS = false) or the
// same map with row / col pointing at a shared-memory copy (kS = true, fused kernel in fn_beam.cuh).
template <bool kS>
__device__ __forceinline__ void reset_env(const ResetArgs& a, const MapDev& mp, const ColScratch& scratch,
                                          const int e, const int lane, BeamPose* pose_copy = nullptr) {
    const int n = a.n;
    const double rho = (double)mp.rho;
    const float two_pi_f = 6.28318530717958647692f, pi_f = 3.14159265358979323846f;
    const float dmin2 = __fmul_rn(a.task.dmin, a.task.dmin), dmax2 = __fmul_rn(a.task.dmax, a.task.dmax);
    int r0 = 0, c0 = 0, rh = mp.H, cw = mp.W;
    if (a.regions.n > 0) { const int4 R = a.regions.rects[e % a.regions.n]; r0 = R.x; c0 = R.y; rh = R.z; cw = R.w; }
    const float X0 = (float)((double)c0 * rho), Xe = (float)((double)cw * rho);
    const float Y0 = (float)((double)r0 * rho), Ye = (float)((double)rh * rho);
    const unsigned long long sigma = a.seeds[e];
    // ---- start pose: attempts k = 0..255, 32 at a time
    float x = 0.f, y = 0.f, psi = 0.f;
    double sp = 0.0, cp = 1.0;
    bool ok = false;
    for (int chunk = 0; chunk < kMaxAttempts / 32 && !ok; ++chunk) {
        const unsigned long long k = (unsigned long long)(chunk * 32 + lane);
        const float xk = __fmaf_rn(u24_at(sigma, 3ull * k), Xe, X0);
        const float yk = __fmaf_rn(u24_at(sigma, 3ull * k + 1ull), Ye, Y0);
        const float pk = __fmaf_rn(u24_at(sigma, 3ull * k + 2ull), two_pi_f, -pi_f);
        double sk, ck;
        sincos((double)pk, &sk, &ck);
        Window w = footprint_window<kS>(mp, scratch.verts, a.robot.V, (double)xk, (double)yk, ck, sk);
        // attempts after the first one that is free without any further test cannot win: skip their tests
        const unsigned free_m = __ballot_sync(0xffffffffu, w.status == 0);
        if (free_m && lane > __ffs(free_m) - 1) w.status = 1;
        // One-sided pre-test: a point inside the footprint whose cell is occupied proves a collision.
        // Most random start poses that collide do so deeply, so few attempts need the exact test.
        if (w.status == 2) {
            bool hit = false;
            for (int q = 0; q < a.robot.n_samples && !hit; q += 4) {
                bool h4 = false;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const double2 f = a.robot.samples[min(q + u, a.robot.n_samples - 1)];
                    const int j = __double2int_rd(((double)xk + ck * f.x - sk * f.y) * mp.inv_rho);
                    const int i = __double2int_rd(((double)yk + sk * f.x + ck * f.y) * mp.inv_rho);
                    h4 |= occ_global<kS>(mp, i, j);
                }
                hit = h4;
            }
            if (hit) w.status = 1;
        }
        const bool col = resolve_collisions<kS>(mp, a.robot, w, (double)xk, (double)yk, ck, sk, scratch);
        const unsigned acc_m = __ballot_sync(0xffffffffu, !col);
        ok = acc_m != 0u;
        const int src = ok ? __ffs(acc_m) - 1 : 31;           // exhausted: keep the last candidate
        x = __shfl_sync(0xffffffffu, xk, src); y = __shfl_sync(0xffffffffu, yk, src);
        psi = __shfl_sync(0xffffffffu, pk, src);
        sp = __shfl_sync(0xffffffffu, sk, src); cp = __shfl_sync(0xffffffffu, ck, src);
    }
    bool fail = !ok;
    // ---- goal: attempts m = 0..255, 32 at a time
    float gx = x, gy = y;
    ok = false;
    for (int chunk = 0; chunk < kMaxAttempts / 32 && !ok; ++chunk) {
        const unsigned long long m = (unsigned long long)(chunk * 32 + lane);
        const float ua = __fmaf_rn(2.0f, u24_at(sigma, 768ull + 2ull * m), -1.0f);
        const float ub = __fmaf_rn(2.0f, u24_at(sigma, 768ull + 2ull * m + 1ull), -1.0f);
        const float gxm = __fmaf_rn(ua, a.task.dmax, x);
        const float gym = __fmaf_rn(ub, a.task.dmax, y);
        const float ddx = __fsub_rn(gxm, x), ddy = __fsub_rn(gym, y);
        const float d2 = __fadd_rn(__fmul_rn(ddx, ddx), __fmul_rn(ddy, ddy));
        bool okm = d2 >= dmin2 && d2 <= dmax2;
        if (okm) {
            const int j = __double2int_rd((double)gxm / rho), i = __double2int_rd((double)gym / rho);
            okm = i >= r0 && j >= c0 && i < r0 + rh && j < c0 + cw && !occ_global<kS>(mp, i, j);
        }
        const unsigned okb = __ballot_sync(0xffffffffu, okm);
        ok = okb != 0u;
        const int src = ok ? __ffs(okb) - 1 : 31;
        gx = __shfl_sync(0xffffffffu, gxm, src); gy = __shfl_sync(0xffffffffu, gym, src);
    }
    fail = fail || !ok;
    if (lane == 0) {
        const double gdx = (double)gx - (double)x, gdy = (double)gy - (double)y;
        const float d = (float)sqrt(gdx * gdx + gdy * gdy);
        const float alpha = (float)wrap_pi(atan2(gdy, gdx) - (double)psi);
        a.states[0 * n + e] = x; a.states[1 * n + e] = y; a.states[2 * n + e] = psi;
        a.states[3 * n + e] = 0.f; a.states[4 * n + e] = 0.f; a.states[5 * n + e] = 0.f;
        a.states[6 * n + e] = gx; a.states[7 * n + e] = gy;
        a.d_prev[e] = d;
        a.ep_step[e] = 0;
        if (a.out_goal_obs) { a.out_goal_obs[e] = d; a.out_goal_obs[n + e] = alpha; }
        const BeamPose bp = make_pose<kS>(mp, a.robot, x, y, psi, cp, sp);
        a.poses[e] = bp;
        write_more_poses<kS>(mp, a.robot, a.poses, n, e, x, y, psi, cp, sp);
        if (pose_copy) *pose_copy = bp;                            // (fused kernel: a copy in shared memory)
        if (a.ring) {
            const unsigned long long head = *a.ring_head_dev;
            float* row = a.ring + ((head + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
            const int B = a.robot.B;
            row[B] = d; row[B + 1] = alpha; row[B + 2] = 0.f; row[B + 3] = 0.f; row[B + 4] = 0.f;
        }
        if (a.fail_out) a.fail_out[e] = fail ? 1 : 0;            // (prepared ahead: counted when it is applied)
        else {
            atomicAdd(&a.counters[kResets], 1ull);
            if (fail) atomicAdd(&a.counters[kResetFail], 1ull);
        }
    }
}

// The stores of reset_env for env e from a prepared reset (one thread): a = the arguments of the fn_reset call.
// _early: what belongs to the SIM and the step no longer touches once its outcome warps have finished (episode
// bookkeeping, counters); _late: what the step uses until it completes (the sensing pose its beams are cast from, the
// ring head) and everything that is the CALLER'S -- state planes and goal observation: fn_step hands them out as the
// pre-reset observation, so a kernel of the caller between fn_step and fn_reset may still be reading them when this
// kernel becomes resident (a reader that releases its dependents early); they are loaded before the dependency wait
// (HeldState) and stored after it.  The prepared values are read past L1 (written by a kernel that may still be running).
__device__ __forceinline__ void reset_apply_early(const ResetArgs& a, const PreparedReset& pr, const int e) {
    a.d_prev[e] = __ldcg(pr.d_prev + e);
    a.ep_step[e] = 0;
    atomicAdd(&a.counters[kResets], 1ull);
    atomicAdd(&a.counters[kResetsPrepared], 1ull);
    if (__ldcg(pr.fail + e)) atomicAdd(&a.counters[kResetFail], 1ull);
}
struct HeldState {                       // prepared state planes and goal observation read before they may be stored
    int e;                               // -1: none
    float st[8], g[2];
};
__device__ __forceinline__ HeldState reset_state_held(const ResetArgs& a, const PreparedReset& pr, const int e) {
    HeldState h;
    h.e = e;
    const int n = a.n;
#pragma unroll
    for (int k = 0; k < 8; ++k) h.st[k] = __ldcg(pr.states + k * n + e);
    h.g[0] = __ldcg(pr.goal_obs + e); h.g[1] = __ldcg(pr.goal_obs + n + e);
    return h;
}
__device__ __forceinline__ void reset_state_store(const ResetArgs& a, const HeldState& h) {
    if (h.e < 0) return;
    const int n = a.n;
#pragma unroll
    for (int k = 0; k < 8; ++k) a.states[k * n + h.e] = h.st[k];
    if (a.out_goal_obs) { a.out_goal_obs[h.e] = h.g[0]; a.out_goal_obs[n + h.e] = h.g[1]; }
}
struct HeldPose {                        // a prepared sensing pose read before it may be stored
    int e;                               // -1: none
    uint4 v[sizeof(BeamPose) / 16];
};
__device__ __forceinline__ HeldPose reset_pose_held(const ResetArgs& a, const PreparedReset& pr, const int e) {
    HeldPose h;
    h.e = e;
    const uint4* src = reinterpret_cast<const uint4*>(pr.poses + e);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(BeamPose) / 16); ++k) h.v[k] = __ldcg(src + k);
    asm volatile("prefetch.global.L2 [%0];" ::"l"(a.poses + e));
    return h;
}
__device__ __forceinline__ void reset_pose_store(const ResetArgs& a, const HeldPose& h) {
    if (h.e < 0) return;
    uint4* dst = reinterpret_cast<uint4*>(a.poses + h.e);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(BeamPose) / 16); ++k) dst[k] = h.v[k];
}
__device__ __forceinline__ void reset_apply_late(const ResetArgs& a, const PreparedReset& pr, const int e, const bool copy_pose = true) {
    const int n = a.n;
    if (copy_pose) {
        const uint4* src = reinterpret_cast<const uint4*>(pr.poses + e);
        uint4* dst = reinterpret_cast<uint4*>(a.poses + e);
#pragma unroll
        for (int k = 0; k < (int)(sizeof(BeamPose) / 16); ++k) dst[k] = src[k];
    }
    if (a.ring) {
        const float d = pr.goal_obs[e], alpha = pr.goal_obs[n + e];
        const unsigned long long head = *a.ring_head_dev;
        float* row = a.ring + ((head + (unsigned long long)e) % a.ring_cap) * (size_t)a.ring_row;
        const int B = a.robot.B;
        row[B] = d; row[B + 1] = alpha; row[B + 2] = 0.f; row[B + 3] = 0.f; row[B + 4] = 0.f;
    }
}

__global__ void __launch_bounds__(kResetWarps * 32) reset_kernel(ResetArgs a) {
    extern __shared__ __align__(16) uint8_t s_dyn[];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const ColScratch scratch = col_scratch(s_dyn + (size_t)wib * col_scratch_bytes(a.robot.V), a.robot.V);
    for (int k = lane; k < a.robot.V; k += 32) { scratch.verts[k] = a.robot.verts[k]; scratch.nxt[k] = a.robot.nxt[k]; }
    __syncwarp();
    griddep_wait();                                                // the list comes from the compaction kernel
    griddep_launch_dependents();
    if (blockIdx.x == 0 && threadIdx.x == 0) *a.beam_task_counter = 0u;
    if (a.list_par_dev) { const int q = *a.list_par_dev ^ 1; a.list += (size_t)q * a.n; a.count_dev += q; }
    const int count = *a.count_dev;
    for (int li = blockIdx.x * kResetWarps + wib; li < count; li += gridDim.x * kResetWarps)
        reset_env<false>(a, a.map, scratch, a.list[li], lane);
}

// ---------------------------------------------------------------- observe-all support: poses from states
struct PoseArgs {
    MapDev map;
    RobotDev robot;
    int n;
    const float* states;
    float* out_goal_obs;         // or NULL
    BeamPose* poses;
    unsigned* beam_task_counter; // zeroed here for the beam kernel that follows
};
__global__ void __launch_bounds__(256) pose_from_state_kernel(PoseArgs a) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e == 0) *a.beam_task_counter = 0u;
    if (e >= a.n) return;
    const int n = a.n;
    const float x = a.states[e], y = a.states[n + e], psi = a.states[2 * n + e];
    double s, c;
    sincos((double)psi, &s, &c);
    write_pose(a.map, a.robot, a.poses, a.n, e, x, y, psi, c, s);
    if (a.out_goal_obs) {
        const double gdx = (double)a.states[6 * n + e] - (double)x, gdy = (double)a.states[7 * n + e] - (double)y;
        a.out_goal_obs[e] = (float)sqrt(gdx * gdx + gdy * gdy);
        a.out_goal_obs[n + e] = (float)wrap_pi(atan2(gdy, gdx) - (double)psi);
    }
}

// ---------------------------------------------------------------- evaluation mode: fixed start-goal cases
// PAPER.md:88 "Each batch assigns fixed start-goal cases to separate environments".  states holds the start
// poses (planes 0-2) and goals (planes 6, 7) of the first n_cases envs; velocities are zeroed, the episode
// state re-seeded, the completion masks cleared (slots >= n_cases are inactive) and the sensing poses set.
struct EvalBeginArgs {
    PoseArgs pose;
    float* states;
    float* d_prev;
    int* ep_step;
    uint8_t* outcome;
    float* ret;
    int n_cases;
};
__global__ void __launch_bounds__(256) eval_begin_kernel(EvalBeginArgs a) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e == 0) *a.pose.beam_task_counter = 0u;
    const int n = a.pose.n;
    if (e >= n) return;
    const float x = a.states[e], y = a.states[n + e], psi = a.states[2 * n + e];
    a.states[3 * n + e] = 0.f; a.states[4 * n + e] = 0.f; a.states[5 * n + e] = 0.f;
    double s, c;
    sincos((double)psi, &s, &c);
    write_pose(a.pose.map, a.pose.robot, a.pose.poses, a.pose.n, e, x, y, psi, c, s);
    const double gdx = (double)a.states[6 * n + e] - (double)x, gdy = (double)a.states[7 * n + e] - (double)y;
    const float d = (float)sqrt(gdx * gdx + gdy * gdy);
    if (a.pose.out_goal_obs) {
        a.pose.out_goal_obs[e] = d;
        a.pose.out_goal_obs[n + e] = (float)wrap_pi(atan2(gdy, gdx) - (double)psi);
    }
    a.d_prev[e] = d;
    a.ep_step[e] = 0;
    a.outcome[e] = e < a.n_cases ? 0 : 4;
    a.ret[e] = 0.f;
}

}  // namespace fn

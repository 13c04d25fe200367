/*
 * fn_oracle.c -- CPU ORACLE for the FlashNav batched simulator step (arxiv/paper_2606_15846).
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded, fp64 C.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load this library.  It shares
 * no code, header, table or helper with the CUDA path under paper_2606_15846_b200/ and neither
 * imports the other.
 *
 * What it computes (citations are PAPER.md lines; "SURVEY 8(c)" = /root/repo/SURVEY.md section 8(c),
 * whose readings are restated in DESIGN.md "Readings of the paper"):
 *   O1/O2  action clip + planar motion update for (v_x, w) / (v_x, v_y, w) body-frame commands
 *          (integrator = exact constant-twist arc, reading G1).
 *   O3     footprint collision: Eq. (2), taken to the limit of a zero footprint
 *          sampling interval = closed polygon vs closed occupied cell; outside the map = collision.
 *   O4     range sensing: PAPER.md:86 fixed-step beam samples taken to the limit of a zero step =
 *          distance to the first occupied cell along the beam; no hit => max range.
 *   O5     goal distance d and direction alpha relative to the robot.
 *   O6     reward Eq. (1), PAPER.md:69-72 (r_success=10, r_collision=-10, c_1=2) and termination.
 *   O7     reset of masked envs (PAPER.md:86, :199 say THAT envs are reset; the sampling rule is
 *          reading G16 -- "parity unpinned" by the paper, pinned by invariants only).
 *   O9     transition row for the replay ring (BASELINE.json config 5).
 *   O11    uniform replay sampling: readings G22 in DESIGN.md.
 *   O10    clearance features, Eq. (3) and their sector min-pooling:
 *          SURVEY 8(f) NEXT-1.  The sector layout is reading G21.
 *   plus the paper's own two approximations as brute-force cross-checks:
 *          fno_ranges_fixed_step and fno_collision_sampled (Eq. (2)).
 *
 * Conventions (reading G7): map-frame origin at the outer corner of cell (row 0, col 0); x grows with
 * column, y with row; cell (i,j) = [j rho,(j+1) rho) x [i rho,(i+1) rho); linear index i*W + j;
 * anything outside [0,W) x [0,H) is occupied (PAPER.md:123 for collision; reading G6 for beams).
 * All inputs are fp32 and are widened exactly to fp64; outputs are rounded once to fp32.
 *
 * Pins (tests/test_oracle_*.py): motion -> closed-form arc / composition; ranges -> empty map, wall,
 * single-cell slab closed form, the paper's fixed-step march, 90-degree symmetry; collision -> interval
 * overlap, notch case, Eq. (2) sampling, point-in-polygon supersampling; reward ->
 * Eq. (1) constants.  UNPINNED by the paper: reset distribution, goal tolerance, episode limit.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define FNO_PI 3.14159265358979323846

enum { FNO_DRIVE_DIFF = 0, FNO_DRIVE_OMNI = 1 };

/* ------------------------------------------------------------------ map lookup (G6, G7) */

static int occ_at(const uint8_t* occ, int H, int W, long i, long j) {
    if (i < 0 || j < 0 || i >= H || j >= W) return 1;          /* outside the map => occupied */
    return occ[(size_t)i * (size_t)W + (size_t)j] != 0;
}

static double wrap_pi(double a) {                               /* to [-pi, pi) (G4) */
    double r = fmod(a + FNO_PI, 2.0 * FNO_PI);
    if (r < 0.0) r += 2.0 * FNO_PI;
    return r - FNO_PI;
}

/* ------------------------------------------------------------------ O1 + O2: clip and motion
 * commands (v_x, w) [diff] or (v_x, v_y, w) [omni], body frame, "within the configured
 * bounds".  Reading G1: the pose is advanced by the exact constant-twist SE(2) step
 *   th = w dt,  A = sin(th)/th,  C = (1-cos th)/th = sin^2(th/2)/(th/2)
 *   body displacement = dt (A v_x - C v_y, C v_x + A v_y),  p' = p + R(psi) * body displacement,
 *   psi' = wrap(psi + th),  v' = clipped command.
 * states: SoA planes [8][n] = x, y, psi, vx, vy, w, gx, gy.  actions: [n][A].
 */
/* acc = NULL or [3] = a_x, a_y, a_w maxima (reading G2, NEXT-3: U "contains velocity and acceleration
 * limits"): the clipped command is further limited to the previous applied velocity
 * +- a_max dt, both bounds single fp32 fused operations (velocities are stored in fp32); +inf = no limit. */
static float slew(float u, float v_prev, float a_max, float dt) {
    if (!(a_max < INFINITY)) return u;
    const float lo = fmaf(-a_max, dt, v_prev), hi = fmaf(a_max, dt, v_prev);
    return fminf(fmaxf(u, lo), hi);
}

void fno_motion_acc(int drive, const float* lim /*[6]*/, const float* acc /*[3] or NULL*/, float dt_f, int n,
                    const float* s_in, const float* actions, float* s_out) {
    const int A = (drive == FNO_DRIVE_DIFF) ? 2 : 3;
    const double dt = (double)dt_f;
    for (int e = 0; e < n; ++e) {
        double x = s_in[0 * n + e], y = s_in[1 * n + e], psi = s_in[2 * n + e];
        double vx = actions[e * A + 0], vy = 0.0, w;
        if (drive == FNO_DRIVE_DIFF) { w = actions[e * A + 1]; }
        else { vy = actions[e * A + 1]; w = actions[e * A + 2]; }
        /* O1: clamp each component to U's velocity limits */
        vx = fmin(fmax(vx, (double)lim[0]), (double)lim[1]);
        if (drive == FNO_DRIVE_OMNI) vy = fmin(fmax(vy, (double)lim[2]), (double)lim[3]);
        w = fmin(fmax(w, (double)lim[4]), (double)lim[5]);
        if (acc) {
            vx = (double)slew((float)vx, s_in[3 * n + e], acc[0], dt_f);
            if (drive == FNO_DRIVE_OMNI) vy = (double)slew((float)vy, s_in[4 * n + e], acc[1], dt_f);
            w = (double)slew((float)w, s_in[5 * n + e], acc[2], dt_f);
        }
        /* O2 */
        double th = w * dt, Ac, Cc;
        if (fabs(th) < 1e-8) { Ac = 1.0 - th * th / 6.0; Cc = th / 2.0; }
        else { double sh = sin(0.5 * th); Ac = sin(th) / th; Cc = sh * sh / (0.5 * th); }
        double bx = dt * (Ac * vx - Cc * vy), by = dt * (Cc * vx + Ac * vy);
        double c = cos(psi), s = sin(psi);
        s_out[0 * n + e] = (float)(x + c * bx - s * by);
        s_out[1 * n + e] = (float)(y + s * bx + c * by);
        s_out[2 * n + e] = (float)wrap_pi(psi + th);
        s_out[3 * n + e] = (float)vx;
        s_out[4 * n + e] = (float)vy;
        s_out[5 * n + e] = (float)w;
        s_out[6 * n + e] = s_in[6 * n + e];
        s_out[7 * n + e] = s_in[7 * n + e];
    }
}

void fno_motion(int drive, const float* lim /*[6]*/, float dt_f, int n,
                const float* s_in, const float* actions, float* s_out) {
    fno_motion_acc(drive, lim, NULL, dt_f, n, s_in, actions, s_out);
}

/* ------------------------------------------------------------------ O5: goal observation
 * d_t = goal distance, alpha_t = goal direction relative to the robot heading.
 */
void fno_goal_obs(int n, const float* x, const float* y, const float* psi,
                  const float* gx, const float* gy, float* d_out, float* alpha_out) {
    for (int e = 0; e < n; ++e) {
        double dx = (double)gx[e] - (double)x[e], dy = (double)gy[e] - (double)y[e];
        d_out[e] = (float)sqrt(dx * dx + dy * dy);
        alpha_out[e] = (float)wrap_pi(atan2(dy, dx) - (double)psi[e]);
    }
}

/* ------------------------------------------------------------------ O6: reward and termination
 * Eq. (1): r = r_collision on collision; r_success when the goal is reached WITHOUT
 * collision; c_1 (d_t - d_{t+1}) otherwise.  done = collision | reached | episode limit | forced.
 * d_prev and ep_step are per-env episode state, updated in place (reading G17: d_prev is from the
 * same episode; reset re-seeds it).
 */
void fno_reward_done(int n, const float* d_new, const uint8_t* collision, const uint8_t* forced,
                     float goal_tol, int max_episode_steps, float r_success, float r_collision,
                     float c_progress, float* d_prev, int32_t* ep_step, float* reward,
                     uint8_t* done) {
    for (int e = 0; e < n; ++e) {
        int c = collision[e] != 0;
        int reached = (double)d_new[e] < (double)goal_tol;
        double r;
        if (c) r = (double)r_collision;
        else if (reached) r = (double)r_success;
        else r = (double)c_progress * ((double)d_prev[e] - (double)d_new[e]);
        int limit = (max_episode_steps > 0) && (ep_step[e] + 1 >= max_episode_steps);
        reward[e] = (float)r;
        done[e] = (uint8_t)(c || reached || limit || (forced && forced[e]));
        d_prev[e] = d_new[e];
        ep_step[e] += 1;
    }
}

/* ------------------------------------------------------------------ O3: footprint collision
 * Eq. (2): c = OR over footprint samples s of M(R(psi) s + p); a collision is
 * detected if any sample lies in an occupied cell or outside the map.  The footprint "interior and
 * boundary are sampled at a configured spatial resolution".  Taking the sampling
 * interval to zero, the sample set becomes the closed polygon region, so
 *   c = 1  iff  some occupied-or-outside cell's closed unit square meets the closed polygon region.
 * Square vs simple polygon: they meet iff (some polygon edge meets the closed square) or (the
 * square's centre is inside the polygon).  [If no edge meets the square, the square lies wholly
 * inside or wholly outside the polygon, and its centre decides which.]
 *
 * Near-tie rule, margin eps in cell units: a cell ROBUSTLY intersects if an edge meets
 * the square shrunk by eps per side or the centre is inside; it is ROBUSTLY disjoint if no edge meets
 * the square grown by eps and the centre is outside.  The flag is ambiguous iff no occupied cell
 * robustly intersects and some occupied cell is not robustly disjoint.
 */

/* closed segment P->Q vs closed box, by slab clipping of the segment parameter (Liang-Barsky) */
static int seg_meets_box(double px, double py, double qx, double qy,
                         double xlo, double xhi, double ylo, double yhi) {
    double t0 = 0.0, t1 = 1.0;
    double dx = qx - px, dy = qy - py;
    double p[4] = { -dx, dx, -dy, dy };
    double q[4] = { px - xlo, xhi - px, py - ylo, yhi - py };
    for (int k = 0; k < 4; ++k) {
        if (p[k] == 0.0) { if (q[k] < 0.0) return 0; }
        else {
            double r = q[k] / p[k];
            if (p[k] < 0.0) { if (r > t1) return 0; if (r > t0) t0 = r; }
            else            { if (r < t0) return 0; if (r < t1) t1 = r; }
        }
    }
    return t0 <= t1;
}

/* even-odd crossing rule; polygon may be CW or CCW, collinear vertices allowed (G13) */
static int point_in_poly(int V, const double* vx, const double* vy, double px, double py) {
    int inside = 0;
    for (int a = 0, b = V - 1; a < V; b = a++) {
        if ((vy[a] > py) != (vy[b] > py)) {
            double xc = (vx[b] - vx[a]) * (py - vy[a]) / (vy[b] - vy[a]) + vx[a];
            if (px < xc) inside = !inside;
        }
    }
    return inside;
}

#define FNO_MAX_V 256

/* one pose -> flag (return value) and ambiguity (*amb) */
static int collision_one(const uint8_t* occ, int H, int W, double rho, int V, const float* fp_xy,
                         double x, double y, double psi, double eps, int* amb) {
    double vx[FNO_MAX_V], vy[FNO_MAX_V];
    double c = cos(psi), s = sin(psi);
    double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    for (int k = 0; k < V; ++k) {
        double fx = fp_xy[2 * k], fy = fp_xy[2 * k + 1];
        vx[k] = (x + c * fx - s * fy) / rho;                    /* cell units */
        vy[k] = (y + s * fx + c * fy) / rho;
        xmin = fmin(xmin, vx[k]); xmax = fmax(xmax, vx[k]);
        ymin = fmin(ymin, vy[k]); ymax = fmax(ymax, vy[k]);
    }
    long j0 = (long)floor(xmin - eps), j1 = (long)floor(xmax + eps);
    long i0 = (long)floor(ymin - eps), i1 = (long)floor(ymax + eps);
    int flag = 0, robust = 0, near = 0;
    for (long i = i0; i <= i1; ++i) for (long j = j0; j <= j1; ++j) {
        if (!occ_at(occ, H, W, i, j)) continue;
        double xl = (double)j, yl = (double)i;
        int in_c = point_in_poly(V, vx, vy, xl + 0.5, yl + 0.5);
        int e_exact = 0, e_shrunk = 0, e_grown = 0;
        for (int a = 0, b = V - 1; a < V; b = a++) {
            if (seg_meets_box(vx[b], vy[b], vx[a], vy[a], xl - eps, xl + 1 + eps, yl - eps, yl + 1 + eps)) {
                e_grown = 1;
                if (seg_meets_box(vx[b], vy[b], vx[a], vy[a], xl, xl + 1, yl, yl + 1)) e_exact = 1;
                if (seg_meets_box(vx[b], vy[b], vx[a], vy[a], xl + eps, xl + 1 - eps, yl + eps, yl + 1 - eps)) e_shrunk = 1;
            }
        }
        if (e_exact || in_c) flag = 1;
        if (e_shrunk || in_c) robust = 1;
        if (e_grown || in_c) near = 1;
    }
    if (amb) *amb = (!robust && near);
    return flag;
}

/* Footprints that are a UNION of polygons ("polygon(s)", :129 "For a union of polygons, the
 * minimum distance over its components is used").  The vertex list is the components'
 * vertex lists one after the other; fno_set_footprint_components gives their sizes (C = 0 or 1: one
 * polygon).  The union collides iff some component does; it robustly collides iff some component robustly
 * does, and is near a collision iff some component is -- hence the ambiguity rule below.  The oracle is
 * single-threaded test infrastructure, so this setting is simply file-scope state.
 */
static int g_ncomp = 0;
static int g_comp[FNO_MAX_V];

void fno_set_footprint_components(int C, const int32_t* sizes) {
    g_ncomp = (C > 1 && C <= FNO_MAX_V) ? C : 0;
    for (int c = 0; c < g_ncomp; ++c) g_comp[c] = sizes[c];
}

static int collision_union(const uint8_t* occ, int H, int W, double rho, int V, const float* fp_xy,
                           double x, double y, double psi, double eps, int* amb) {
    if (g_ncomp <= 1) return collision_one(occ, H, W, rho, V, fp_xy, x, y, psi, eps, amb);
    int flag = 0, robust = 0, near = 0, off = 0;
    for (int c = 0; c < g_ncomp; ++c) {
        int a = 0;
        const int f = collision_one(occ, H, W, rho, g_comp[c], fp_xy + 2 * off, x, y, psi, eps, &a);
        flag |= f;
        robust |= (f && !a);
        near |= (f || a);
        off += g_comp[c];
    }
    (void)V;
    if (amb) *amb = (!robust && near);
    return flag;
}

void fno_collision(const uint8_t* occ, int H, int W, float res, int V, const float* fp_xy, int n,
                   const float* x, const float* y, const float* psi, double eps,
                   uint8_t* flag, uint8_t* amb) {
    for (int e = 0; e < n; ++e) {
        int a = 0;
        flag[e] = (uint8_t)collision_union(occ, H, W, (double)res, V, fp_xy, x[e], y[e], psi[e], eps, &a);
        if (amb) amb[e] = (uint8_t)a;
    }
}

/* Eq. (2) exactly as the paper states it: sample the footprint interior and
 * boundary at spacing h (metres, body frame), cache the point set, OR the occupancy of the cells the
 * transformed samples fall in.  Cross-check only: sampled => exact always; exact-by-a-margin => sampled.
 * Interior: body-frame lattice points inside the polygon; boundary: points every <= h along each edge.
 */
void fno_collision_sampled(const uint8_t* occ, int H, int W, float res, int V, const float* fp_xy,
                           double h, int n, const float* x, const float* y, const float* psi,
                           uint8_t* flag) {
    double bx[FNO_MAX_V], by[FNO_MAX_V];
    double xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    for (int k = 0; k < V; ++k) {
        bx[k] = fp_xy[2 * k]; by[k] = fp_xy[2 * k + 1];
        xmin = fmin(xmin, bx[k]); xmax = fmax(xmax, bx[k]);
        ymin = fmin(ymin, by[k]); ymax = fmax(ymax, by[k]);
    }
    size_t cap = 1024, np_ = 0;
    double* P = (double*)malloc(cap * 2 * sizeof(double));
#define PUSH(px_, py_) do { if (np_ == cap) { cap *= 2; P = (double*)realloc(P, cap * 2 * sizeof(double)); } \
                            P[2 * np_] = (px_); P[2 * np_ + 1] = (py_); ++np_; } while (0)
    for (double yy = ymin; yy <= ymax; yy += h)
        for (double xx = xmin; xx <= xmax; xx += h)
            if (point_in_poly(V, bx, by, xx, yy)) PUSH(xx, yy);
    for (int a = 0, b = V - 1; a < V; b = a++) {
        double ex = bx[a] - bx[b], ey = by[a] - by[b];
        int m = (int)ceil(sqrt(ex * ex + ey * ey) / h);
        if (m < 1) m = 1;
        for (int k = 0; k <= m; ++k) PUSH(bx[b] + ex * k / m, by[b] + ey * k / m);
    }
#undef PUSH
    double rho = (double)res;
    for (int e = 0; e < n; ++e) {
        double c = cos((double)psi[e]), s = sin((double)psi[e]);
        int f = 0;
        for (size_t k = 0; k < np_ && !f; ++k) {
            double wx = ((double)x[e] + c * P[2 * k] - s * P[2 * k + 1]) / rho;
            double wy = ((double)y[e] + s * P[2 * k] + c * P[2 * k + 1]) / rho;
            f = occ_at(occ, H, W, (long)floor(wy), (long)floor(wx));
        }
        flag[e] = (uint8_t)f;
    }
    free(P);
}

/* ------------------------------------------------------------------ O4: range sensing
 * "Range sensing uses fixed-step samples along each beam."  With step Delta the range is
 * the first sample distance whose cell is occupied; as Delta -> 0 this becomes
 *   r = rho * inf{ t >= 0 : M(cell(o + t d)) = 1 },  capped at r_max,   no hit => r_max
 * with o the sensor origin in cell units and d = (cos phi, sin phi), phi = psi + s_psi + theta_j.
 * The infimum is found by walking the grid cell by cell (Amanatides-Woo): the next vertical /
 * horizontal cell boundary along the beam is at parameter t_x = (b_x - o_x)/d_x, t_y = (b_y - o_y)/d_y,
 * each computed DIRECTLY from the boundary coordinate (never accumulated); the smaller one is crossed
 * first.  The first occupied (or outside-map) cell entered at t_hit < r_max/rho gives
 *   range = t_hit * rho, hit = i*W + j  (-2 if that cell is outside the map);
 * origin already in an occupied cell => range 0; otherwise range = r_max, hit = -1.
 *
 * Near-tie rule, eps in cells: a beam is ambiguous iff, up to and including the entry
 * into the hit cell, it passes within eps of a lattice corner whose four surrounding cells do not all
 * have the same occupancy, or |t_hit - r_max/rho| < eps (also: an occupied cell first entered within
 * eps beyond r_max/rho), or the origin lies within eps of a cell edge separating different occupancy.
 * sensor[3] = (s_x, s_y, s_psi) body-frame sensor placement (reading G8), NULL = 0.
 * visits (optional, per beam): number of cells the walk entered (workload statistics only).
 */
static int corner_mixed(const uint8_t* occ, int H, int W, long cx, long cy) {
    int a = occ_at(occ, H, W, cy - 1, cx - 1), b = occ_at(occ, H, W, cy - 1, cx);
    int c = occ_at(occ, H, W, cy, cx - 1),     d = occ_at(occ, H, W, cy, cx);
    return !(a == b && b == c && c == d);
}

static void ray_one(const uint8_t* occ, int H, int W, double rho, double ox, double oy, double phi,
                    double T, double rmax, double eps, float* range, int32_t* hit, uint8_t* amb,
                    int32_t* visits) {
    double dx = cos(phi), dy = sin(phi);
    long j = (long)floor(ox), i = (long)floor(oy);
    int ambiguous = 0, nvis = 1;
    /* origin within eps of an edge separating different occupancy */
    {
        int here = occ_at(occ, H, W, i, j);
        double fx = ox - (double)j, fy = oy - (double)i;
        if (fx < eps && occ_at(occ, H, W, i, j - 1) != here) ambiguous = 1;
        if (1.0 - fx < eps && occ_at(occ, H, W, i, j + 1) != here) ambiguous = 1;
        if (fy < eps && occ_at(occ, H, W, i - 1, j) != here) ambiguous = 1;
        if (1.0 - fy < eps && occ_at(occ, H, W, i + 1, j) != here) ambiguous = 1;
        if (here) {
            *range = 0.0f;
            *hit = (i >= 0 && j >= 0 && i < H && j < W) ? (int32_t)(i * W + j) : -2;
            if (amb) *amb = (uint8_t)ambiguous;
            if (visits) *visits = nvis;
            return;
        }
    }
    long sx = dx > 0.0 ? 1 : -1, sy = dy > 0.0 ? 1 : -1;
    double bx = dx > 0.0 ? (double)(j + 1) : (double)j;         /* next vertical boundary   */
    double by = dy > 0.0 ? (double)(i + 1) : (double)i;         /* next horizontal boundary */
    double tx = dx != 0.0 ? (bx - ox) / dx : INFINITY;
    double ty = dy != 0.0 ? (by - oy) / dy : INFINITY;
    for (;;) {
        double t;
        int step_x = 0, step_y = 0;
        if (tx < ty) { t = tx; step_x = 1; }
        else if (ty < tx) { t = ty; step_y = 1; }
        else { t = tx; step_x = step_y = 1; }                   /* exactly through a corner */
        /* nearest lattice corner on the boundary line being crossed; perpendicular distance to the beam */
        if (t < T + eps) {
            if (step_x) {
                double yc = oy + t * dy; long cy = (long)floor(yc + 0.5), cx = (long)bx;
                double dist = fabs(((double)cx - ox) * dy - ((double)cy - oy) * dx);
                if (dist < eps && corner_mixed(occ, H, W, cx, cy)) ambiguous = 1;
            }
            if (step_y) {
                double xc = ox + t * dx; long cx = (long)floor(xc + 0.5), cy = (long)by;
                double dist = fabs(((double)cx - ox) * dy - ((double)cy - oy) * dx);
                if (dist < eps && corner_mixed(occ, H, W, cx, cy)) ambiguous = 1;
            }
        }
        if (step_x) { j += sx; bx += (double)sx; tx = (bx - ox) / dx; }
        if (step_y) { i += sy; by += (double)sy; ty = (by - oy) / dy; }
        if (t >= T) {                                           /* cell entered at or beyond r_max */
            if (t - T < eps && occ_at(occ, H, W, i, j)) ambiguous = 1;
            *range = (float)rmax; *hit = -1;
            break;
        }
        ++nvis;
        if (occ_at(occ, H, W, i, j)) {
            if (T - t < eps) ambiguous = 1;
            *range = (float)(t * rho);
            *hit = (i >= 0 && j >= 0 && i < H && j < W) ? (int32_t)(i * W + j) : -2;
            break;
        }
    }
    if (amb) *amb = (uint8_t)ambiguous;
    if (visits) *visits = nvis;
}

void fno_ranges(const uint8_t* occ, int H, int W, float res, int B, const float* angles,
                float max_range, const float* sensor /*[3] or NULL*/, int n,
                const float* x, const float* y, const float* psi, double eps,
                float* ranges /*[n][B]*/, int32_t* hit /*[n][B] or NULL*/,
                uint8_t* amb /*[n][B] or NULL*/, int32_t* visits /*[n][B] or NULL*/) {
    const double rho = (double)res, rmax = (double)max_range, T = rmax / rho;
    const double s0 = sensor ? (double)sensor[0] : 0.0, s1 = sensor ? (double)sensor[1] : 0.0,
                 s2 = sensor ? (double)sensor[2] : 0.0;
    for (int e = 0; e < n; ++e) {
        double c = cos((double)psi[e]), s = sin((double)psi[e]);
        double ox = ((double)x[e] + c * s0 - s * s1) / rho;
        double oy = ((double)y[e] + s * s0 + c * s1) / rho;
        for (int b = 0; b < B; ++b) {
            size_t k = (size_t)e * (size_t)B + (size_t)b;
            double phi = (double)psi[e] + s2 + (double)angles[b];
            int32_t h;
            ray_one(occ, H, W, rho, ox, oy, phi, T, rmax, eps, &ranges[k], &h,
                    amb ? &amb[k] : NULL, visits ? &visits[k] : NULL);
            if (hit) hit[k] = h;
        }
    }
}

/* A robot with several range sensors ("S defines sensor placement and range-sensing parameters";
 * PAPER.md:125 "using the sensor placement in the robot specification").  Sensor k has its own
 * placement (s_x, s_y, s_psi) in the body frame, beam table (B_k angles) and maximum range; the observation row of
 * an env is the concatenation of the sensors' ranges in sensor order (B = sum of B_k).  Every beam is the plain
 * definition of O4 from its own sensor's origin.
 */
void fno_ranges_multi(const uint8_t* occ, int H, int W, float res, int K, const int32_t* Bk /*[K]*/,
                      const float* angles /*[sum Bk]*/, const float* max_range /*[K]*/, const float* sensors /*[K][3]*/,
                      int n, const float* x, const float* y, const float* psi, double eps,
                      float* ranges /*[n][B]*/, int32_t* hit /*[n][B] or NULL*/, uint8_t* amb /*[n][B] or NULL*/) {
    const double rho = (double)res;
    size_t B = 0;
    for (int k = 0; k < K; ++k) B += (size_t)Bk[k];
    for (int e = 0; e < n; ++e) {
        const double c = cos((double)psi[e]), s = sin((double)psi[e]);
        size_t off = 0;
        for (int k = 0; k < K; ++k) {
            const double s0 = (double)sensors[3 * k], s1 = (double)sensors[3 * k + 1], s2 = (double)sensors[3 * k + 2];
            const double rmax = (double)max_range[k], T = rmax / rho;
            const double ox = ((double)x[e] + c * s0 - s * s1) / rho;      /* sensor origin in the map frame, in cells */
            const double oy = ((double)y[e] + s * s0 + c * s1) / rho;
            for (int b = 0; b < Bk[k]; ++b) {
                const size_t i = (size_t)e * B + off + (size_t)b;
                const double phi = (double)psi[e] + s2 + (double)angles[off + (size_t)b];
                int32_t h;
                ray_one(occ, H, W, rho, ox, oy, phi, T, rmax, eps, &ranges[i], &h, amb ? &amb[i] : NULL, NULL);
                if (hit) hit[i] = h;
            }
            off += (size_t)Bk[k];
        }
    }
}

/* The paper's own definition: fixed-step samples along each beam, first sample at t = 0
 * (reading G5), step `delta` metres; the range is the distance of the first sample that falls in an
 * occupied (or outside-map) cell; no such sample below r_max => r_max.  Cross-check only.
 */
void fno_ranges_fixed_step(const uint8_t* occ, int H, int W, float res, int B, const float* angles,
                           float max_range, double delta, int n, const float* x, const float* y,
                           const float* psi, float* ranges) {
    const double rho = (double)res, rmax = (double)max_range;
    for (int e = 0; e < n; ++e) for (int b = 0; b < B; ++b) {
        double phi = (double)psi[e] + (double)angles[b], dx = cos(phi), dy = sin(phi);
        double r = rmax;
        for (long k = 0; ; ++k) {
            double t = (double)k * delta;
            if (t >= rmax) break;
            double px = ((double)x[e] + t * dx) / rho, py = ((double)y[e] + t * dy) / rho;
            if (occ_at(occ, H, W, (long)floor(py), (long)floor(px))) { r = t; break; }
        }
        ranges[(size_t)e * B + b] = (float)r;
    }
}

/* ------------------------------------------------------------------ O7: reset of masked envs
 * PAPER.md:86 "When episodes end, only the corresponding environments are reset"; "their
 * environments are reset to start new episodes".  The paper gives no sampling rule; this is reading
 * G16 (BASELINE.json config 1: "Start poses uniform in free space, goals 3-8 m away"), PARITY UNPINNED.
 *
 * Random numbers: counter-based SplitMix64 (Steele, Lea, Flood 2014 finaliser): draw c of seed sigma is
 *   z = sigma + (c+1) * 0x9E3779B97F4A7C15;  z = (z ^ z>>30) * 0xBF58476D1CE4E5B9;
 *   z = (z ^ z>>27) * 0x94D049BB133111EB;    z ^ z>>31
 * i.e. the (c+1)-th output of a SplitMix64 stream seeded with sigma.  Uniform u = (z >> 40) * 2^-24,
 * exact in fp32.  Start attempt k = 0..255 uses draws 3k, 3k+1, 3k+2; goal attempt m = 0..255 uses
 * draws 768+2m, 768+2m+1.  All fp32 operations below are single, separately rounded operations.
 */
uint64_t fno_splitmix64(uint64_t sigma, uint64_t c) {
    uint64_t z = sigma + (c + 1u) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
static float u24(uint64_t sigma, uint64_t c) {
    return (float)(fno_splitmix64(sigma, c) >> 40) * 5.9604644775390625e-08f;   /* 2^-24 */
}

#define FNO_MAX_ATTEMPTS 256

static int goal_cell_ok(const uint8_t* occ, int H, int W, long r0, long c0, long rh, long cw, long i, long j) {
    if (i < r0 || j < c0 || i >= r0 + rh || j >= c0 + cw) return 0;
    return !occ_at(occ, H, W, i, j);
}

/* states [8][n] updated in place for masked envs; d_prev/ep_step re-seeded; amb/fail optional. */
void fno_reset(const uint8_t* occ, int H, int W, float res, int V, const float* fp_xy,
               int n_regions, const int32_t* regions /*[n_regions][4] or NULL*/,
               float goal_dist_min, float goal_dist_max, int n, const uint8_t* mask,
               const uint64_t* seeds, double eps, float* states, float* d_prev, int32_t* ep_step,
               uint8_t* amb /*[n] or NULL*/, uint8_t* failed /*[n] or NULL*/) {
    const double rho = (double)res;
    const float two_pi_f = 6.28318530717958647692f, pi_f = 3.14159265358979323846f;
    const float dmin2 = goal_dist_min * goal_dist_min, dmax2 = goal_dist_max * goal_dist_max;
    for (int e = 0; e < n; ++e) {
        if (amb) amb[e] = 0;
        if (failed) failed[e] = 0;
        if (!mask[e]) continue;
        long r0 = 0, c0 = 0, rh = H, cw = W;
        if (n_regions > 0 && regions) {
            const int32_t* R = regions + 4 * (e % n_regions);
            r0 = R[0]; c0 = R[1]; rh = R[2]; cw = R[3];
        }
        const float X0 = (float)((double)c0 * rho), Xe = (float)((double)cw * rho);
        const float Y0 = (float)((double)r0 * rho), Ye = (float)((double)rh * rho);
        const uint64_t sigma = seeds[e];
        int ambiguous = 0, fail = 0;
        float x = 0, y = 0, psi = 0;
        int ok = 0;
        for (int k = 0; k < FNO_MAX_ATTEMPTS && !ok; ++k) {
            x = fmaf(u24(sigma, 3u * k), Xe, X0);
            y = fmaf(u24(sigma, 3u * k + 1u), Ye, Y0);
            psi = fmaf(u24(sigma, 3u * k + 2u), two_pi_f, -pi_f);
            int a = 0;
            ok = !collision_union(occ, H, W, rho, V, fp_xy, x, y, psi, eps, &a);
            ambiguous |= a;
        }
        if (!ok) fail = 1;
        float gx = x, gy = y;
        ok = 0;
        for (int m = 0; m < FNO_MAX_ATTEMPTS && !ok; ++m) {
            float a = fmaf(2.0f, u24(sigma, 768u + 2u * m), -1.0f);       /* exact */
            float b = fmaf(2.0f, u24(sigma, 768u + 2u * m + 1u), -1.0f);
            gx = fmaf(a, goal_dist_max, x);
            gy = fmaf(b, goal_dist_max, y);
            float ddx = gx - x, ddy = gy - y;
            float p = ddx * ddx, q = ddy * ddy;
            float d2 = p + q;
            if (!(d2 >= dmin2 && d2 <= dmax2)) continue;
            double cx = (double)gx / rho, cy = (double)gy / rho;
            long j = (long)floor(cx), i = (long)floor(cy);
            ok = goal_cell_ok(occ, H, W, r0, c0, rh, cw, i, j);
            /* goal point within eps of a cell edge across which acceptability differs */
            double fx = cx - (double)j, fy = cy - (double)i;
            long dj0 = fx < eps ? -1 : 0, dj1 = (1.0 - fx) < eps ? 1 : 0;
            long di0 = fy < eps ? -1 : 0, di1 = (1.0 - fy) < eps ? 1 : 0;
            for (long di = di0; di <= di1; ++di) for (long dj = dj0; dj <= dj1; ++dj)
                if (goal_cell_ok(occ, H, W, r0, c0, rh, cw, i + di, j + dj) != ok) ambiguous = 1;
        }
        if (!ok) fail = 1;
        states[0 * n + e] = x;  states[1 * n + e] = y;  states[2 * n + e] = psi;
        states[3 * n + e] = 0;  states[4 * n + e] = 0;  states[5 * n + e] = 0;
        states[6 * n + e] = gx; states[7 * n + e] = gy;
        double ex = (double)gx - (double)x, ey = (double)gy - (double)y;
        d_prev[e] = (float)sqrt(ex * ex + ey * ey);
        ep_step[e] = 0;
        if (amb) amb[e] = (uint8_t)ambiguous;
        if (failed) failed[e] = (uint8_t)fail;
    }
}

/* ------------------------------------------------------------------ O9: replay-ring row
 * PAPER.md:84 "transitions are written directly to a GPU-resident circular replay buffer";
 * BASELINE.json config 5: "(obs, action, reward, done) in fp32".  Row layout (reading G18):
 *   [ranges(B), d, alpha, v_x, v_y, w, action(A), reward, done]  with obs = the observation the action
 * was chosen from.  slot = (head + e) mod capacity.
 * done is a code (reading G18, revised): 0 = the episode goes on, 1 = it TERMINATED (collision or goal reached:
 * PAPER.md:69-72, the cases Eq. (1) rewards), 2 = it was TRUNCATED (step limit or a forced reset, no terminal
 * event).  PAPER.md:86 keeps the pre-reset observation as the next observation of such a row; this ring's next
 * observation of a done row is the post-reset one (G22), so a learner must not bootstrap from it -- with the code it
 * can tell the rows whose bootstrap is legitimately zero (1) from the rows it has to leave out (2).
 * fno_done_code gives the code from what the step reports.
 */
uint8_t fno_done_code(uint8_t done, uint8_t collision, float d, float goal_tol) {
    if (!done) return 0;
    return (collision || d < goal_tol) ? 1 : 2;
}

void fno_ring_append(float* ring, uint64_t capacity, uint64_t head, int n, int B, int A,
                     const float* obs_ranges /*[n][B]*/, const float* obs_goal /*[2][n]*/,
                     const float* obs_vel /*[3][n]*/, const float* actions /*[n][A]*/,
                     const float* reward, const uint8_t* done) {
    const size_t row = (size_t)B + 5 + (size_t)A + 2;
    for (int e = 0; e < n; ++e) {
        float* r = ring + (size_t)((head + (uint64_t)e) % capacity) * row;
        memcpy(r, obs_ranges + (size_t)e * B, (size_t)B * sizeof(float));
        r[B + 0] = obs_goal[0 * n + e]; r[B + 1] = obs_goal[1 * n + e];
        r[B + 2] = obs_vel[0 * n + e];  r[B + 3] = obs_vel[1 * n + e]; r[B + 4] = obs_vel[2 * n + e];
        for (int a = 0; a < A; ++a) r[B + 5 + a] = actions[(size_t)e * A + a];
        r[B + 5 + A] = reward[e];
        r[B + 6 + A] = (float)done[e];                             /* the code: 0, 1 or 2 */
    }
}

/* ------------------------------------------------------------------ O10: clearance features (NEXT-1)
 * "Each valid range endpoint e_{t,j} ... is expressed in the body frame using the
 * sensor placement in the robot specification.  Its nonnegative distance to the occupied footprint is
 * delta_{t,j} = min_{f in F} ||e_{t,j} - f||_2 (3).  For polygonal footprints, this distance is computed
 * directly from the boundary segments and is set to zero for points inside the occupied region. ...
 * Distances are capped at the sensor range and pooled by taking the minimum within each angular sector.
 * Beams without a valid hit are assigned the maximum range before pooling."  (also PAPER.md:67)
 * Readings: valid <=> range < max_range (G10); endpoint = s_xy + r (cos, sin)(theta_j + s_psi) (G8);
 * sector of beam j = floor(j n_sectors / B), i.e. n_sectors groups of consecutive beams in table order
 * (G21: the paper gives neither the sector count nor its layout).
 */
static double point_segment_dist(double px, double py, double ax, double ay, double bx, double by) {
    const double ex = bx - ax, ey = by - ay, l2 = ex * ex + ey * ey;
    double t = l2 > 0.0 ? ((px - ax) * ex + (py - ay) * ey) / l2 : 0.0;
    if (t < 0.0) t = 0.0;
    if (t > 1.0) t = 1.0;
    return hypot(px - (ax + t * ex), py - (ay + t * ey));
}

static int point_in_polygon(double px, double py, int V, const float* fp_xy) {   /* even-odd rule */
    int in = 0;
    for (int k = 0, j = V - 1; k < V; j = k++) {
        const double ax = fp_xy[2 * j], ay = fp_xy[2 * j + 1], bx = fp_xy[2 * k], by = fp_xy[2 * k + 1];
        if ((ay > py) != (by > py) && px < ax + (py - ay) * (bx - ax) / (by - ay)) in = !in;
    }
    return in;
}

/* Eq. (3) for one body-frame point and one polygon */
static double polygon_distance(int V, const float* fp_xy, double px, double py) {
    if (point_in_polygon(px, py, V, fp_xy)) return 0.0;
    double d = INFINITY;
    for (int k = 0, j = V - 1; k < V; j = k++) {
        const double dk = point_segment_dist(px, py, fp_xy[2 * j], fp_xy[2 * j + 1], fp_xy[2 * k], fp_xy[2 * k + 1]);
        if (dk < d) d = dk;
    }
    return d;
}

/* ... and for the footprint: "For a union of polygons, the minimum distance over its components" */
double fno_footprint_distance(int V, const float* fp_xy, double px, double py) {
    if (g_ncomp <= 1) return polygon_distance(V, fp_xy, px, py);
    double d = INFINITY;
    int off = 0;
    for (int c = 0; c < g_ncomp; ++c) {
        const double dc = polygon_distance(g_comp[c], fp_xy + 2 * off, px, py);
        if (dc < d) d = dc;
        off += g_comp[c];
    }
    return d;
}

void fno_clearance_features(int V, const float* fp_xy, int B, const float* angles, const float* sensor /*[3] or NULL*/,
                            float max_range, int n_sectors, int n, const float* ranges /*[n][B]*/,
                            float* delta /*[n][B] or NULL*/, float* z /*[n][n_sectors]*/) {
    const double s0 = sensor ? (double)sensor[0] : 0.0, s1 = sensor ? (double)sensor[1] : 0.0,
                 s2 = sensor ? (double)sensor[2] : 0.0;
    const double rmax = (double)max_range;
    for (int e = 0; e < n; ++e) {
        for (int k = 0; k < n_sectors; ++k) z[(size_t)e * n_sectors + k] = max_range;
        for (int j = 0; j < B; ++j) {
            const double r = (double)ranges[(size_t)e * B + j];
            double d = rmax;                                          /* no valid hit: the maximum range */
            if (r < rmax) {
                const double phi = (double)angles[j] + s2;
                d = fno_footprint_distance(V, fp_xy, s0 + r * cos(phi), s1 + r * sin(phi));
                if (d > rmax) d = rmax;                               /* capped at the sensor range */
            }
            if (delta) delta[(size_t)e * B + j] = (float)d;
            const int k = (int)(((long long)j * n_sectors) / B);
            if ((float)d < z[(size_t)e * n_sectors + k]) z[(size_t)e * n_sectors + k] = (float)d;
        }
    }
}

/* ------------------------------------------------------------------ O11: replay sampling (NEXT-2)
 * "Each replay batch contains U x B transitions sampled uniformly from replay and divided
 * into U minibatches of size B."  Readings (G22): the rows that can be sampled are the COMPLETED transitions
 * still in the ring.  With `total` rows appended so far, head = total mod capacity is the slot of env 0's
 * PENDING row: the n_envs rows [head, head + n_envs) already hold the observation the next actions will be
 * chosen from, but action, reward and done of a transition that has not happened (stale values of the row
 * they overwrote once the ring has wrapped), so they are excluded: valid = min(total, capacity - n_envs) rows,
 * the oldest at slot head - valid (mod capacity).  Sample i of a batch draws s_i = floor(w_i valid / 2^64)
 * with w_i = SplitMix64(seed, i) (the counter-based generator of O7) and takes slot (head - valid + s_i) mod
 * capacity (before the ring is that full: slot s_i); the batch row is the ring row (obs, action, reward, done)
 * as stored; the next observation is the obs part of the SAME env's next row, slot + n_envs (mod capacity),
 * which the step that completed the row has already written (for the newest transitions that is the pending
 * row).  For a done transition that is the post-reset observation unless terminal observations are kept: see
 * fno_terminal_save and the sampler below.
 */
uint64_t fno_sample_slot(uint64_t seed, uint64_t i, uint64_t filled) {
    const uint64_t w = fno_splitmix64(seed, i);
    return (uint64_t)(((unsigned __int128)w * (unsigned __int128)filled) >> 64);
}

uint64_t fno_ring_valid(uint64_t capacity, uint64_t total, int n_envs) {
    const uint64_t room = capacity > (uint64_t)n_envs ? capacity - (uint64_t)n_envs : 0;
    return total < room ? total : room;
}
/* Terminal observations ("Observations before reset are retained as next observations in replay,
 * while reset observations are returned to the collector").  In the ring the next observation of a row is the obs
 * part of the same env's next row, and a reset overwrites that pending row with the reset observation.  So, before a
 * reset touches it, the pending row's obs part [ranges(B), d, alpha, v_x, v_y, w] -- the observation the step left
 * behind, i.e. the terminal one -- is copied into a second, smaller ring of `t_cap` terminal entries (t_cap >=
 * n_envs), for every listed env whose last completed row (slot head - n_envs + e, global row id total - n_envs + e)
 * has a done code != 0 and is not kept yet.  term_idx[slot] = the entry of that ring row, term_id[entry] = the
 * global id of the row the entry belongs to, *term_head = the entries ever written (entry = index mod t_cap, reused
 * in order).  The entries written by the resets that follow ONE step form a batch; batch_start = *term_head when
 * that step ended (term_start[entry]); a batch is given up as a whole as soon as a later write reuses any of its
 * entries, i.e. an entry is kept while its id matches and *term_head <= term_start[entry] + t_cap.  (So what is
 * kept does not depend on the order in which the envs of one reset are listed.)  list = the envs being reset.
 */
static int fno_terminal_kept(uint64_t slot, uint64_t g, uint64_t t_cap, const int32_t* term_idx, const uint64_t* term_id,
                             const uint64_t* term_start, uint64_t term_head) {
    const int32_t t = term_idx[slot];
    return t >= 0 && term_id[t] == g && term_head <= term_start[t] + t_cap;
}
void fno_terminal_save(const float* ring, uint64_t capacity, uint64_t total, int n_envs, int B, int A,
                       const int32_t* list, int count, float* term /*[t_cap][B+5]*/, uint64_t t_cap,
                       int32_t* term_idx /*[capacity]*/, uint64_t* term_id /*[t_cap]*/, uint64_t* term_start /*[t_cap]*/,
                       uint64_t* term_head, uint64_t batch_start) {
    const size_t row = (size_t)B + 5 + (size_t)A + 2, obs = (size_t)B + 5;
    if (total < (uint64_t)n_envs) return;                        /* no step has completed a row yet */
    const uint64_t head = total % capacity;
    for (int k = 0; k < count; ++k) {
        const uint64_t e = (uint64_t)list[k];
        const uint64_t c = (head + capacity - (uint64_t)n_envs + e) % capacity;      /* the env's last completed row */
        const uint64_t g = total - (uint64_t)n_envs + e;
        if (ring[c * row + (size_t)B + 6 + (size_t)A] == 0.0f) continue;             /* the episode did not end */
        if (fno_terminal_kept(c, g, t_cap, term_idx, term_id, term_start, *term_head)) continue;   /* kept already */
        const uint64_t entry = *term_head % t_cap;
        *term_head += 1;
        memcpy(term + entry * obs, ring + ((head + e) % capacity) * row, obs * sizeof(float));
        term_id[entry] = g;
        term_start[entry] = batch_start;
        term_idx[c] = (int32_t)entry;
    }
}

/* The sampler with terminal observations.  term == NULL: no terminal ring.  For a row with done code != 0 whose
 * terminal entry is still there, the next observation is that entry (the pre-reset observation); otherwise it is
 * the obs part of the env's next row as before (the post-reset observation).  The done field of the SAMPLED copy
 * says which: 0 running, 1 terminated (bootstrap masked, next observation irrelevant), 2 truncated with its true
 * next observation delivered, 3 truncated but the observation is gone (or no terminal ring): not to be
 * bootstrapped from.  Ring rows themselves hold 0, 1, 2 (fno_done_code).
 */
void fno_ring_sample(const float* ring, uint64_t capacity, uint64_t total, int n_envs, int B, int A,
                     uint64_t seed, int n_samples, float* out_rows /*[n_samples][row]*/,
                     float* out_next_obs /*[n_samples][B+5] or NULL*/, int64_t* out_slots /*or NULL*/,
                     const float* term, uint64_t t_cap, const int32_t* term_idx, const uint64_t* term_id,
                     const uint64_t* term_start, uint64_t term_head) {
    const size_t row = (size_t)B + 5 + (size_t)A + 2, obs = (size_t)B + 5;
    const uint64_t valid = fno_ring_valid(capacity, total, n_envs), head = total % capacity;
    if (valid == 0) return;
    for (int i = 0; i < n_samples; ++i) {
        const uint64_t si = fno_sample_slot(seed, (uint64_t)i, valid);
        const uint64_t slot = (head + capacity - valid + si) % capacity;
        const uint64_t g = total - valid + si;                   /* global id of the sampled row */
        float* out = out_rows + (size_t)i * row;
        memcpy(out, ring + (size_t)slot * row, row * sizeof(float));
        const float* next = ring + (size_t)((slot + (uint64_t)n_envs) % capacity) * row;
        const float code = out[(size_t)B + 6 + (size_t)A];
        if (code != 0.0f) {
            int kept = 0;
            if (term && fno_terminal_kept(slot, g, t_cap, term_idx, term_id, term_start, term_head)) {
                next = term + (size_t)term_idx[slot] * obs;
                kept = 1;
            }
            if (code == 2.0f && !kept) out[(size_t)B + 6 + (size_t)A] = 3.0f;
        }
        if (out_next_obs) memcpy(out_next_obs + (size_t)i * obs, next, obs * sizeof(float));
        if (out_slots) out_slots[i] = (int64_t)slot;
    }
}

/* ------------------------------------------------------------------ O12: evaluation bookkeeping (NEXT-3)
 * "Completion masks record each case once and exclude completed cases from further
 * accumulation of rewards and outcome statistics.  Each case ends when the robot reaches the goal,
 * collides with an obstacle, or reaches the evaluation step limit."  outcome: 0 running, 1 success,
 * 2 collision, 3 step limit, 4 inactive slot; collision has priority over success as in Eq. (1).
 * Called once per vector step with that step's flags for ALL envs; completed cases are left untouched.
 */
void fno_eval_update(int n, const uint8_t* collision, const float* d_new, float goal_tol,
                     const int32_t* ep_step_after, int step_limit, const float* reward,
                     uint8_t* outcome, int32_t* steps, float* ret) {
    for (int e = 0; e < n; ++e) {
        if (outcome[e] != 0) continue;                           /* recorded once; excluded afterwards */
        ret[e] += reward[e];
        int o = 0;
        if (collision[e]) o = 2;
        else if (d_new[e] < goal_tol) o = 1;
        else if (ep_step_after[e] >= step_limit) o = 3;
        if (o) { outcome[e] = (uint8_t)o; steps[e] = ep_step_after[e]; }
    }
}

/* ------------------------------------------------------------------ one whole vector step (3.2)
 * actions -> O1/O2 motion -> O3 collision + O5 goal obs at the new pose -> O6 reward/done ->
 * O4 ranges at the new pose.  Outputs are the PRE-reset (terminal) observations.
 * The caller then applies fno_reset to done envs and recomputes only their observations (O8).
 */
void fno_step(const uint8_t* occ, int H, int W, float res, int V, const float* fp_xy, int B,
              const float* angles, float max_range, int drive, const float* lim, float dt,
              float goal_tol, int max_episode_steps, float r_success, float r_collision,
              float c_progress, int n, float* states /*in/out [8][n]*/, const float* actions,
              const uint8_t* forced, float* d_prev, int32_t* ep_step, float* ranges,
              int32_t* hit, uint8_t* collision, float* goal_obs /*[2][n]*/, float* reward,
              uint8_t* done) {
    float* s2 = (float*)malloc((size_t)8 * n * sizeof(float));
    fno_motion(drive, lim, dt, n, states, actions, s2);
    memcpy(states, s2, (size_t)8 * n * sizeof(float));
    free(s2);
    const float *x = states, *y = states + n, *psi = states + 2 * n, *gx = states + 6 * n, *gy = states + 7 * n;
    fno_collision(occ, H, W, res, V, fp_xy, n, x, y, psi, 0.0, collision, NULL);
    fno_goal_obs(n, x, y, psi, gx, gy, goal_obs, goal_obs + n);
    fno_reward_done(n, goal_obs, collision, forced, goal_tol, max_episode_steps, r_success,
                    r_collision, c_progress, d_prev, ep_step, reward, done);
    fno_ranges(occ, H, W, res, B, angles, max_range, NULL, n, x, y, psi, 0.0, ranges, hit, NULL, NULL);
}

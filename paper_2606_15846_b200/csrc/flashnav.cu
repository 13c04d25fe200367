// flashnav.cu -- host side of the C ABI declared in include/flashnav.h.
// Argument validation, bit-packing and upload of the map, launch configuration.  Every step of the
// hot path runs in the kernels of fn_env.cuh / fn_beam.cuh; nothing here computes simulator results.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>
#include <vector>

#include "../../include/flashnav.h"
#include "fn_beam.cuh"
#include "fn_common.cuh"
#include "fn_env.cuh"
#include "fn_features.cuh"
#include "fn_fixed_step.cuh"
#include "fn_reset_beam.cuh"
#include "fn_step_split.cuh"

using namespace fn;

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
#define FN_CUDA(call)                                                                        \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail(e_ == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA, "%s: %s", \
                        #call, cudaGetErrorString(e_));                                      \
    } while (0)

struct fn_map {
    int H, W;
    float res;
    uint32_t* d_words;       // row-packed copy then column-packed copy, contiguous; then their coarse copies
    size_t n_words;          // the two fine copies, padded to a multiple of 4
    size_t n_words_coarse;   // the two coarse copies (fn_common.cuh, coarse_words), padded to a multiple of 4
    MapDev dev;
    int n_regions;
    int4* d_regions;
    unsigned version;        // bumped by every setter (a reset prepared ahead must see the map it is applied with)
};

constexpr int kMaxSensors = 4;
struct fn_sensor {               // one range sensor: its block of the observation row, table and placement
    int off, B;
    float rmax, sx, sy, spsi;
};
struct fn_robot {
    std::vector<fn_sensor> sensors;  // [0] = the constructor's (beam table, max range) with fn_robot_set_sensor's placement
    int V, B, drive;                 // B = beams of ALL sensors = length of an observation row
    float lim[6];
    float acc[3];
    float rmax;
    float sensor[3];
    std::vector<float> angles;
    std::vector<float> verts;
    double2* d_beam_cs;
    double2* d_verts;
    double2* d_samples;              // interior sample points of the footprint (reset pre-test)
    int n_samples;
    std::vector<int> nxt;            // next vertex within the vertex's component (union of polygons)
    int* d_nxt;
    unsigned version;                // bumped by every setter
};

struct fn_sim {
    const fn_map* map;
    const fn_robot* robot;
    int n;
    fn_task task;
    cudaStream_t stream;
    int num_sms;
    int n_sensors;                   // range sensors of the robot at fn_sim_create (one beam launch and pose set each)
    // device state owned by the sim
    BeamPose* d_poses;
    int* d_list;
    int* d_count;
    float* d_dprev;
    int* d_epstep;
    unsigned long long* d_counters;
    unsigned* d_task_counter;        // beam kernel's dynamic task counter
    uint8_t* d_eval_outcome;         // evaluation mode: completion masks, returns
    float* d_eval_return;
    int eval_mode, eval_limit;
    int* d_done_list;                // [2][n] envs reported done by fn_step (one list per step parity), any order
    int* d_done_count;               // [2] counts, [2] = the parity the NEXT fn_step fills (device-side state)
    int done_avail;                  // 1 = the last fn_step's list has not been consumed by fn_reset(mask = NULL)
    // bound by the caller
    int32_t* aux_hit;
    float* aux_reward;
    float* ring;
    float* feat_z;                   // bound clearance-feature output [n][feat_sectors] or NULL
    int feat_sectors;
    unsigned long long ring_cap;
    unsigned long long* d_ring_head;   // device: slot of env 0's pending ring row
    TerminalDev term;                  // terminal observations (fn_ring_attach_terminal): caller's entries, the sim's index arrays
    int count_words;
    // beam-kernel launch configuration
    bool use_smem;
    size_t beam_smem;
    int beam_grid;
    // fn_reset as one fused kernel (fn_reset_beam.cuh): possible / enabled, its shared bytes and grid
    bool fused_ok, fused_on, fused_force;
    size_t fused_smem;
    int fused_grid;
    // fn_step with the env step split around the beam kernel (fn_step_split.cuh)
    bool split_ok, split_on;
    size_t split_smem;
    int split_grid;
    StepEnd* d_step_end;
    // fn_sim_prepare_reset: the step's outcome warps also run the reset of the envs they report done (prep_ok: the
    // kernels exist for this sim); prep_next = the seeds announced for the coming fn_step, prep_ready = the seeds the
    // buffers were filled with by the last fn_step (with the map / robot versions they were filled under)
    bool prep_ok;
    int prep_grid;
    const uint64_t *prep_next, *prep_ready;
    unsigned prep_map_ver, prep_robot_ver;
    PreparedReset d_prep;
    int* d_prep_epstep;
    unsigned prep_spin;              // polls (64 ns apart) prepared_reset_kernel grants the step's outcome warps before it
                                     // falls back to waiting for the whole step; FLASHNAV_PREP_SPIN overrides (tests: 0)
    // the coarse level in the production beam kernels (one CTA of 1024 threads per SM, fine + coarse copies staged)
    bool coarse_ok, coarse_on, split_ok_c;
    size_t beam_smem_c, split_smem_c;
    int beam_grid_c, split_grid_c;
    // live timing
    int prof;
    std::vector<cudaEvent_t>* ev;    // triples per fn_step (e0 env e1 beam e2), pairs per fn_reset
    std::vector<int>* ev_kind;       // 0 = step triple start, 1 = reset pair start
    // device staging for fn_step_host (lazily allocated)
    float *stg_states, *stg_actions, *stg_ranges, *stg_gobs;
    uint8_t *stg_mask, *stg_col;
    unsigned long long* stg_seeds;
    // fn_step_host_begin / _end: two slots of device staging and events, one copy stream
    struct HostSlot {
        float *ranges, *gobs, *states, *actions;
        uint8_t *mask, *col;
        unsigned long long* seeds;
        cudaEvent_t ev_ready, ev_done;
        bool busy;
    } hslot[2];
    cudaStream_t copy_stream;
    bool pipe_init, pipe_states;     // slots allocated; the device holds the current states
};

extern "C" const char* fn_last_error(void) { return g_err; }
extern "C" const char* fn_version(void) { return "flashnav-b200 0.1 (sm_100a)"; }

extern "C" void fn_task_default(fn_task* t) {
    if (!t) return;
    t->goal_tol_m = 0.3f; t->max_episode_steps = 0; t->goal_dist_min_m = 3.0f; t->goal_dist_max_m = 8.0f;
    t->r_success = 10.0f; t->r_collision = -10.0f; t->c_progress = 2.0f;
}

// ------------------------------------------------------------------------------------------ map
extern "C" int fn_map_create(const uint8_t* bitmap, int H, int W, float res, fn_map** out) {
    if (!bitmap || !out) return fail(FN_ERR_INVALID_ARG, "fn_map_create: NULL argument");
    if (H <= 0 || W <= 0 || H > 32768 || W > 32768) return fail(FN_ERR_INVALID_ARG, "fn_map_create: H, W must be in 1..32768");
    if (!std::isfinite(res) || res <= 0.0f) return fail(FN_ERR_INVALID_ARG, "fn_map_create: resolution must be finite and > 0");
    // Layout (fn_common.cuh): per copy L + 4 lines of nw + 4 words; frame, guards, pads and the bits
    // beyond a line's length are ones ("outside the map is occupied").
    const int nwR = (W + 31) / 32, nwC = (H + 31) / 32;
    const int sR = nwR + 4, sC = nwC + 4;
    const size_t rowWords = (size_t)(H + 2 * kLineGuard) * sR, colWords = (size_t)(W + 2 * kLineGuard) * sC;
    const size_t total = (rowWords + colWords + 3) / 4 * 4;
    std::vector<uint32_t> words(total, 0xffffffffu);
    for (int i = 0; i < H; ++i) {
        uint32_t* line = &words[(size_t)(i + kLineGuard) * sR + (kCellShift >> 5)];
        for (int k = 0; k < nwR; ++k) {
            uint32_t w = 0;
            for (int b = 0; b < 32; ++b) {
                const int j = 32 * k + b;
                if (j >= W || bitmap[(size_t)i * W + j]) w |= 1u << b;
            }
            line[k] = w;
        }
    }
    for (int j = 0; j < W; ++j) {
        uint32_t* line = &words[rowWords + (size_t)(j + kLineGuard) * sC + (kCellShift >> 5)];
        for (int k = 0; k < nwC; ++k) {
            uint32_t w = 0;
            for (int b = 0; b < 32; ++b) {
                const int i = 32 * k + b;
                if (i >= H || bitmap[(size_t)i * W + j]) w |= 1u << b;
            }
            line[k] = w;
        }
    }
    // Coarse level (north_star "coarse block-occupancy level for empty-space skipping"; fn_common.cuh): one line
    // per PAIR of physical lines 2g, 2g + 1 = the OR of the two, stored with twice the line stride.
    const size_t cR = coarse_words(H, sR), cC = coarse_words(W, sC);
    const size_t total_c = (cR + cC + 3) / 4 * 4;
    words.resize(total + total_c, 0xffffffffu);
    for (int copy = 0; copy < 2; ++copy) {
        const int L = copy ? W : H, st = copy ? sC : sR;
        const uint32_t* fine = &words[copy ? rowWords : 0];
        uint32_t* coarse = &words[total + (copy ? cR : 0)];
        for (int p = 0; p < L + 2 * kLineGuard; ++p)
            for (int k = 0; k < st; ++k) {
                uint32_t& w = coarse[(size_t)(p >> 1) * 2 * st + k];
                w = (p & 1) ? (w | fine[(size_t)p * st + k]) : fine[(size_t)p * st + k];
            }
    }
    fn_map* m = new (std::nothrow) fn_map();
    if (!m) return fail(FN_ERR_OOM, "fn_map_create: host allocation failed");
    m->H = H; m->W = W; m->res = res; m->n_words = total; m->n_words_coarse = total_c; m->n_regions = 0; m->d_regions = nullptr; m->d_words = nullptr;
    cudaError_t e = cudaMalloc(&m->d_words, words.size() * sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMemcpy(m->d_words, words.data(), words.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        if (m->d_words) cudaFree(m->d_words);
        delete m;
        return fail(e == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA, "fn_map_create: %s", cudaGetErrorString(e));
    }
    m->dev.row = m->d_words; m->dev.col = m->d_words + rowWords;
    m->dev.H = H; m->dev.W = W; m->dev.nwR = nwR; m->dev.nwC = nwC; m->dev.strideR = sR; m->dev.strideC = sC;
    m->dev.rho = res; m->dev.inv_rho = 1.0 / (double)res;
    *out = m;
    return FN_OK;
}

extern "C" int fn_map_set_regions(fn_map* m, int n, const int32_t* rects) {
    if (!m || n < 0 || (n > 0 && !rects)) return fail(FN_ERR_INVALID_ARG, "fn_map_set_regions: bad argument");
    for (int k = 0; k < n; ++k) {
        const int32_t* r = rects + 4 * k;
        if (r[0] < 0 || r[1] < 0 || r[2] <= 0 || r[3] <= 0 || r[0] + r[2] > m->H || r[1] + r[3] > m->W)
            return fail(FN_ERR_INVALID_ARG, "fn_map_set_regions: rect %d outside the map", k);
    }
    if (m->d_regions) { cudaFree(m->d_regions); m->d_regions = nullptr; }
    m->n_regions = 0;
    if (n > 0) {
        FN_CUDA(cudaMalloc(&m->d_regions, (size_t)n * sizeof(int4)));
        FN_CUDA(cudaMemcpy(m->d_regions, rects, (size_t)n * sizeof(int4), cudaMemcpyHostToDevice));
        m->n_regions = n;
    }
    ++m->version;
    return FN_OK;
}

extern "C" int fn_map_destroy(fn_map* m) {
    if (!m) return FN_OK;
    if (m->d_words) cudaFree(m->d_words);
    if (m->d_regions) cudaFree(m->d_regions);
    delete m;
    return FN_OK;
}

// ------------------------------------------------------------------------------------------ robot
// Up to kMaxSamples points strictly inside the footprint polygon (body frame), on a regular grid over
// its bounding box.  A sample whose map cell is occupied proves a collision (the converse does not hold),
// which lets fn_reset discard most colliding start-pose attempts without the exact polygon test.
constexpr int kMaxSamples = 32;
static std::vector<double2> interior_samples(const std::vector<float>& v, const std::vector<int>& nxt, int V) {
    double x0 = 1e300, x1 = -1e300, y0 = 1e300, y1 = -1e300;
    for (int k = 0; k < V; ++k) {
        x0 = std::fmin(x0, v[2 * k]); x1 = std::fmax(x1, v[2 * k]);
        y0 = std::fmin(y0, v[2 * k + 1]); y1 = std::fmax(y1, v[2 * k + 1]);
    }
    std::vector<double2> pts;
    for (int g : {6, 8, 12, 16}) {
        pts.clear();
        for (int a = 0; a < g; ++a)
            for (int b = 0; b < g; ++b) {
                const double px = x0 + (x1 - x0) * (a + 0.5) / g, py = y0 + (y1 - y0) * (b + 0.5) / g;
                bool in = false, in_c = false;                     // inside ANY component (even-odd per component)
                double dmin = 1e300;
                for (int j = 0; j < V; ++j) {                      // edge j -> nxt[j]
                    const int k = nxt[j];
                    const double ax = v[2 * j], ay = v[2 * j + 1], bx = v[2 * k], by = v[2 * k + 1];
                    if ((ay > py) != (by > py) && px < ax + (py - ay) * (bx - ax) / (by - ay)) in_c = !in_c;
                    if (k <= j) { in = in || in_c; in_c = false; }
                    const double ex = bx - ax, ey = by - ay, l2 = ex * ex + ey * ey;
                    double t = l2 > 0.0 ? ((px - ax) * ex + (py - ay) * ey) / l2 : 0.0;
                    t = std::fmin(1.0, std::fmax(0.0, t));
                    dmin = std::fmin(dmin, std::hypot(px - (ax + t * ex), py - (ay + t * ey)));
                }
                if (in && dmin > 1e-4) pts.push_back(make_double2(px, py));
            }
        if (pts.size() >= 8) break;
    }
    if ((int)pts.size() > kMaxSamples) {                           // thin out evenly
        std::vector<double2> q;
        for (int i = 0; i < kMaxSamples; ++i) q.push_back(pts[(size_t)i * pts.size() / kMaxSamples]);
        pts.swap(q);
    }
    return pts;
}

static int robot_upload(fn_robot* r) {
    std::vector<double2> cs(r->B), vs(r->V);
    for (const fn_sensor& sn : r->sensors)
        for (int j = 0; j < sn.B; ++j) {
            const double a = (double)r->angles[sn.off + j] + (double)sn.spsi;
            cs[sn.off + j] = make_double2(std::cos(a), std::sin(a));
        }
    for (int k = 0; k < r->V; ++k) vs[k] = make_double2((double)r->verts[2 * k], (double)r->verts[2 * k + 1]);
    FN_CUDA(cudaMemcpy(r->d_beam_cs, cs.data(), cs.size() * sizeof(double2), cudaMemcpyHostToDevice));
    FN_CUDA(cudaMemcpy(r->d_verts, vs.data(), vs.size() * sizeof(double2), cudaMemcpyHostToDevice));
    FN_CUDA(cudaMemcpy(r->d_nxt, r->nxt.data(), r->nxt.size() * sizeof(int), cudaMemcpyHostToDevice));
    const std::vector<double2> sp = interior_samples(r->verts, r->nxt, r->V);
    r->n_samples = (int)sp.size();
    if (r->n_samples) FN_CUDA(cudaMemcpy(r->d_samples, sp.data(), sp.size() * sizeof(double2), cudaMemcpyHostToDevice));
    return FN_OK;
}

extern "C" int fn_robot_create_union(const float* fp, const int32_t* comp_sizes, int C, const float* angles, int B,
                                     float rmax, int drive, const float* lim, fn_robot** out) {
    if (!fp || !comp_sizes || !angles || !lim || !out) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: NULL argument");
    if (C < 1) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: a footprint needs >= 1 polygon");
    int V = 0;
    for (int c = 0; c < C; ++c) {
        if (comp_sizes[c] < 3) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: footprint needs >= 3 vertices (per polygon)");
        V += comp_sizes[c];
        if (V > FN_MAX_VERTS) return fail(FN_ERR_UNSUPPORTED, "fn_robot_create: V > FN_MAX_VERTS (%d)", FN_MAX_VERTS);
    }
    if (B < 1) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: B must be >= 1");
    if (!std::isfinite(rmax) || rmax <= 0.0f) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: max range must be finite and > 0");
    if (drive != FN_DRIVE_DIFF && drive != FN_DRIVE_OMNI) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: unknown drive type");
    for (int k = 0; k < 6; k += 2)
        if (!std::isfinite(lim[k]) || !std::isfinite(lim[k + 1]) || lim[k] > lim[k + 1])
            return fail(FN_ERR_INVALID_ARG, "fn_robot_create: velocity limits must be finite with min <= max");
    for (int k = 0; k < 2 * V; ++k) if (!std::isfinite(fp[k])) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: non-finite footprint vertex");
    for (int j = 0; j < B; ++j) if (!std::isfinite(angles[j])) return fail(FN_ERR_INVALID_ARG, "fn_robot_create: non-finite beam angle");
    fn_robot* r = new (std::nothrow) fn_robot();
    if (!r) return fail(FN_ERR_OOM, "fn_robot_create: host allocation failed");
    r->V = V; r->B = B; r->drive = drive; r->rmax = rmax;
    std::memcpy(r->lim, lim, sizeof(r->lim));
    r->sensor[0] = r->sensor[1] = r->sensor[2] = 0.0f;
    r->acc[0] = r->acc[1] = r->acc[2] = INFINITY;
    r->angles.assign(angles, angles + B);
    r->sensors.assign(1, fn_sensor{0, B, rmax, 0.0f, 0.0f, 0.0f});
    r->verts.assign(fp, fp + 2 * V);
    r->nxt.resize(V);
    for (int c = 0, off = 0; c < C; off += comp_sizes[c], ++c)
        for (int k = 0; k < comp_sizes[c]; ++k) r->nxt[off + k] = off + (k + 1 == comp_sizes[c] ? 0 : k + 1);
    r->d_beam_cs = nullptr; r->d_verts = nullptr; r->d_samples = nullptr; r->n_samples = 0; r->d_nxt = nullptr;
    cudaError_t e = cudaMalloc(&r->d_beam_cs, (size_t)B * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc(&r->d_verts, (size_t)V * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc(&r->d_nxt, (size_t)V * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&r->d_samples, (size_t)kMaxSamples * sizeof(double2));
    int st = (e == cudaSuccess) ? robot_upload(r) : fail(e == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA, "fn_robot_create: %s", cudaGetErrorString(e));
    if (st != FN_OK) {
        if (r->d_beam_cs) cudaFree(r->d_beam_cs);
        if (r->d_verts) cudaFree(r->d_verts);
        if (r->d_nxt) cudaFree(r->d_nxt);
        if (r->d_samples) cudaFree(r->d_samples);
        delete r;
        return st;
    }
    *out = r;
    return FN_OK;
}

extern "C" int fn_robot_create(const float* fp, int V, const float* angles, int B, float rmax, int drive,
                               const float* lim, fn_robot** out) {
    const int32_t one = V;
    return fn_robot_create_union(fp, &one, 1, angles, B, rmax, drive, lim, out);
}

extern "C" int fn_robot_set_sensor(fn_robot* r, float sx, float sy, float spsi) {
    if (!r || !std::isfinite(sx) || !std::isfinite(sy) || !std::isfinite(spsi)) return fail(FN_ERR_INVALID_ARG, "fn_robot_set_sensor: bad argument");
    r->sensor[0] = sx; r->sensor[1] = sy; r->sensor[2] = spsi;
    r->sensors[0].sx = sx; r->sensors[0].sy = sy; r->sensors[0].spsi = spsi;
    ++r->version;
    return robot_upload(r);
}

extern "C" int fn_robot_add_sensor(fn_robot* r, const float* angles, int B, float rmax, float sx, float sy, float spsi) {
    if (!r || !angles) return fail(FN_ERR_INVALID_ARG, "fn_robot_add_sensor: NULL argument");
    if (B < 1) return fail(FN_ERR_INVALID_ARG, "fn_robot_add_sensor: B must be >= 1");
    if (!std::isfinite(rmax) || rmax <= 0.0f) return fail(FN_ERR_INVALID_ARG, "fn_robot_add_sensor: max range must be finite and > 0");
    if (!std::isfinite(sx) || !std::isfinite(sy) || !std::isfinite(spsi)) return fail(FN_ERR_INVALID_ARG, "fn_robot_add_sensor: non-finite placement");
    for (int j = 0; j < B; ++j) if (!std::isfinite(angles[j])) return fail(FN_ERR_INVALID_ARG, "fn_robot_add_sensor: non-finite beam angle");
    if ((int)r->sensors.size() >= kMaxSensors) return fail(FN_ERR_UNSUPPORTED, "fn_robot_add_sensor: at most %d sensors", kMaxSensors);
    double2* cs = nullptr;
    cudaError_t e = cudaMalloc(&cs, (size_t)(r->B + B) * sizeof(double2));
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA, "fn_robot_add_sensor: %s", cudaGetErrorString(e));
    cudaFree(r->d_beam_cs);
    r->d_beam_cs = cs;
    r->sensors.push_back(fn_sensor{r->B, B, rmax, sx, sy, spsi});
    r->angles.insert(r->angles.end(), angles, angles + B);
    r->B += B;
    if (rmax > r->rmax) r->rmax = rmax;                            // the robot's largest range (clearance cap, limits)
    ++r->version;
    return robot_upload(r);
}

extern "C" int fn_robot_set_acc_limits(fn_robot* r, const float* acc) {
    if (!r || !acc) return fail(FN_ERR_INVALID_ARG, "fn_robot_set_acc_limits: NULL argument");
    for (int k = 0; k < 3; ++k)
        if (!(acc[k] > 0.0f)) return fail(FN_ERR_INVALID_ARG, "fn_robot_set_acc_limits: limits must be > 0 (+inf = none)");
    for (int k = 0; k < 3; ++k) r->acc[k] = acc[k];
    return FN_OK;
}

extern "C" int fn_robot_destroy(fn_robot* r) {
    if (!r) return FN_OK;
    if (r->d_beam_cs) cudaFree(r->d_beam_cs);
    if (r->d_verts) cudaFree(r->d_verts);
    if (r->d_nxt) cudaFree(r->d_nxt);
    if (r->d_samples) cudaFree(r->d_samples);
    delete r;
    return FN_OK;
}

static RobotDev robot_dev(const fn_robot* r, const fn_map* m) {
    RobotDev d;
    d.beam_cs = r->d_beam_cs; d.verts = r->d_verts; d.nxt = r->d_nxt; d.samples = r->d_samples; d.n_samples = r->n_samples; d.B = r->B; d.V = r->V; d.drive = r->drive;
    d.A = r->drive == FN_DRIVE_DIFF ? 2 : 3;
    for (int k = 0; k < 6; ++k) d.lim[k] = r->lim[k];
    for (int k = 0; k < 3; ++k) d.acc[k] = r->acc[k];
    d.rmax = r->rmax;
    d.T = (double)r->rmax / (double)m->res;
    d.sx = r->sensor[0]; d.sy = r->sensor[1];
    d.n_sensors = (int)r->sensors.size();
    for (int k = 0; k < 4; ++k) { d.sxs[k] = d.sys[k] = 0.0; }
    for (int k = 0; k < d.n_sensors; ++k) { d.sxs[k] = r->sensors[k].sx; d.sys[k] = r->sensors[k].sy; }
    return d;
}
static TaskDev task_dev(const fn_task& t) {
    TaskDev d;
    d.goal_tol = t.goal_tol_m; d.max_episode_steps = t.max_episode_steps; d.dmin = t.goal_dist_min_m;
    d.dmax = t.goal_dist_max_m; d.r_success = t.r_success; d.r_collision = t.r_collision; d.c_progress = t.c_progress;
    return d;
}

// ------------------------------------------------------------------------------------------ sim
// The dynamic shared-memory limit is an attribute of the FUNCTION, not of a sim: it is raised to the device's
// opt-in maximum once, so that sims with different map sizes can live side by side; occupancy is per sim.
constexpr bool kCoarseDefault = false;   // (set by measurement: DESIGN.md 6.1)
template <class K>
static cudaError_t kernel_config(K kernel, int threads, size_t smem, int max_optin, int* blocks_per_sm) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
    if (e != cudaSuccess) return e;
    const int dyn_max = max_optin - (int)fa.sharedSizeBytes;       // static + dynamic <= opt-in maximum
    if ((long long)smem > (long long)dyn_max) { *blocks_per_sm = 0; return cudaSuccess; }
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, kernel, threads, smem);
}
template <bool S, bool C>
static cudaError_t beam_config(size_t smem, int max_optin, int* blocks_per_sm) {
    return kernel_config(beam_kernel<S, C>, kBeamThreads, smem, max_optin, blocks_per_sm);
}

extern "C" int fn_sim_create(const fn_map* map, const fn_robot* robot, int n, const fn_task* task,
                             void* stream, fn_sim** out) {
    if (!map || !robot || !out) return fail(FN_ERR_INVALID_ARG, "fn_sim_create: NULL argument");
    if (n <= 0) return fail(FN_ERR_INVALID_ARG, "fn_sim_create: n_envs must be > 0");
    if ((long long)n * robot->B >= (1ll << 31)) return fail(FN_ERR_UNSUPPORTED, "fn_sim_create: n_envs * B must be < 2^31");
    fn_sim* s = new (std::nothrow) fn_sim();
    if (!s) return fail(FN_ERR_OOM, "fn_sim_create: host allocation failed");
    std::memset(s, 0, sizeof(*s));
    s->map = map; s->robot = robot; s->n = n; s->stream = (cudaStream_t)stream;
    if (task) s->task = *task; else fn_task_default(&s->task);
    s->prep_spin = 1u << 16;                                       // ~4 ms; the flag is normally up before the kernel starts
    if (const char* v = std::getenv("FLASHNAV_PREP_SPIN")) s->prep_spin = (unsigned)std::strtoul(v, nullptr, 10);
    if (!(s->task.goal_dist_min_m >= 0.0f) || !(s->task.goal_dist_max_m >= s->task.goal_dist_min_m)) {
        delete s;
        return fail(FN_ERR_INVALID_ARG, "fn_sim_create: goal distance range must satisfy 0 <= min <= max");
    }
    int dev = 0, max_optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    s->n_sensors = (int)robot->sensors.size();
    if (e == cudaSuccess) e = cudaMalloc(&s->d_poses, (size_t)n * s->n_sensors * sizeof(BeamPose));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_ring_head, 4 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_ring_head, 0, 4 * sizeof(unsigned long long), s->stream);
    if (e == cudaSuccess) e = cudaMalloc(&s->d_list, (size_t)n * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_count, sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_dprev, (size_t)n * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_epstep, (size_t)n * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_counters, kNCounters * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_task_counter, sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_eval_outcome, (size_t)n);
    if (e == cudaSuccess) e = cudaMalloc(&s->d_eval_return, (size_t)n * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_step_end, sizeof(StepEnd));
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_step_end, 0, sizeof(StepEnd), s->stream);
    if (e == cudaSuccess) e = cudaMalloc(&s->d_done_list, 2 * (size_t)n * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_done_count, 3 * sizeof(int));
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_done_count, 0, 3 * sizeof(int), s->stream);
    s->done_avail = 0;
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_task_counter, 0, sizeof(unsigned), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_dprev, 0, (size_t)n * sizeof(float), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_epstep, 0, (size_t)n * sizeof(int), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_counters, 0, kNCounters * sizeof(unsigned long long), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_poses, 0xff, (size_t)n * s->n_sensors * sizeof(BeamPose), s->stream);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(env_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                   (int)col_scratch_bytes(FN_MAX_VERTS));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(reset_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                   (int)(kResetWarps * col_scratch_bytes(FN_MAX_VERTS)));
    if (e == cudaSuccess) {
        // stage the packed map in shared memory when both copies + the beam table fit, else read via L2
        const size_t tab = (size_t)robot->B * sizeof(double2);
        const size_t with_map = tab + map->n_words * sizeof(uint32_t);
        // the shared-memory kernel recovers the line count from the bit offset: needs T + 34 < S / 2
        const double Tc = (double)robot->rmax / (double)map->res;
        const int Smin = 32 * ((map->dev.strideR < map->dev.strideC) ? map->dev.strideR : map->dev.strideC);
        // ... and addresses bits within a copy by the 20-bit integer field of a double in [2^20, 2^21)
        const size_t rowBits = (size_t)(map->H + 2 * kLineGuard) * map->dev.strideR * 32;
        const size_t colBits = (size_t)(map->W + 2 * kLineGuard) * map->dev.strideC * 32;
        s->use_smem = with_map + 8192 <= (size_t)max_optin && Tc + 34.0 < 0.5 * (double)Smin &&   // (8 KB: the kernels' static shared memory)
                      rowBits < (1u << 20) && colBits < (1u << 20);
        s->beam_smem = s->use_smem ? with_map : tab;
        if (s->beam_smem > (size_t)max_optin) {
            fn_sim_destroy(s);
            return fail(FN_ERR_UNSUPPORTED, "fn_sim_create: beam table does not fit in shared memory (B too large)");
        }
        int bps = 0, bps2 = 0;
        if (s->use_smem) { e = beam_config<true, false>(s->beam_smem, max_optin, &bps); if (e == cudaSuccess) e = beam_config<true, true>(s->beam_smem, max_optin, &bps2); }
        else { e = beam_config<false, false>(s->beam_smem, max_optin, &bps); if (e == cudaSuccess) e = beam_config<false, true>(s->beam_smem, max_optin, &bps2); }
        if (bps2 < bps) bps = bps2;
        if (bps < 1) bps = 1;
        s->beam_grid = s->num_sms * bps;
        // the fused reset + beam kernel: the beam kernel's shared memory plus the reset warps' scratch
        s->fused_ok = s->fused_on = false;
        s->fused_smem = fused_smem_bytes(robot->B, (int)map->n_words, robot->V);
        s->fused_grid = 0;
        if (e == cudaSuccess && s->use_smem && s->fused_smem <= (size_t)max_optin) {
            int f0 = 0, f1 = 0;
            e = kernel_config(reset_beam_kernel<false>, kFusedThreads, s->fused_smem, max_optin, &f0);
            if (e == cudaSuccess) e = kernel_config(reset_beam_kernel<true>, kFusedThreads, s->fused_smem, max_optin, &f1);
            if (f1 < f0) f0 = f1;
            // (several sensors: one beam launch per sensor, so the reset and the step keep their own kernels)
            if (e == cudaSuccess && f0 >= 1 && s->n_sensors == 1) { s->fused_ok = s->fused_on = true; s->fused_grid = s->num_sms * f0; }
        }
        // the split step: the beam kernel plus one collision scratch; used when it keeps the beam kernel's occupancy
        s->split_ok = s->split_on = false;
        s->split_smem = step_split_smem_bytes(s->beam_smem, robot->V);
        s->split_grid = 0;
        if (e == cudaSuccess && s->split_smem <= (size_t)max_optin) {
            int f[2] = {0, 0};
            if (s->use_smem) {
                e = kernel_config(step_beam_kernel<true, false>, kBeamThreads, s->split_smem, max_optin, &f[0]);
                if (e == cudaSuccess) e = kernel_config(step_beam_kernel<true, true>, kBeamThreads, s->split_smem, max_optin, &f[1]);
            } else {
                e = kernel_config(step_beam_kernel<false, false>, kBeamThreads, s->split_smem, max_optin, &f[0]);
                if (e == cudaSuccess) e = kernel_config(step_beam_kernel<false, true>, kBeamThreads, s->split_smem, max_optin, &f[1]);
            }
            const int fm = f[0] < f[1] ? f[0] : f[1];
            if (e == cudaSuccess && fm >= 1 && s->num_sms * fm >= s->beam_grid && s->n_sensors == 1) {
                s->split_ok = true; s->split_grid = s->num_sms * fm;
                // one warp per CTA computes the outcomes of the envs its CTA owns, 32 at a time: worth it up to
                // two such batches (measured: C1-C4 3-8 % faster per step, C5 with 222 envs per CTA 4 % slower)
                s->split_on = (n + s->split_grid - 1) / s->split_grid <= 64;
            }
            // ... and its variant that prepares the resets (served by the fused reset kernel)
            // (its fn_reset is prepared_reset_kernel: the production beam kernel's shape)
            s->prep_ok = false;
            if (e == cudaSuccess && s->split_ok && s->use_smem) {
                int fp = 0, fq = 0;
                e = kernel_config(step_beam_kernel<true, false, false, true>, kBeamThreads, s->split_smem, max_optin, &fp);
                if (e == cudaSuccess) e = kernel_config(prepared_reset_kernel, kBeamThreads, s->beam_smem, max_optin, &fq);
                // worth it when the beam casting lasts longer than the chain of a reset (~10 us; the outcome warp runs
                // its resets one after the other): eight rounds of 32 beams per warp (C1's 64 envs: 33 -> 36 us per step)
                const size_t rounds_all = (size_t)n * (((size_t)robot->B + 31) >> 5), warps_all = (size_t)s->split_grid * (kBeamThreads / 32);
                s->prep_ok = e == cudaSuccess && s->num_sms * fp >= s->split_grid && fq >= 1 && rounds_all >= 8 * warps_all;
                s->prep_grid = s->num_sms * fq;
            }
        }
        // the coarse level: fine + coarse copies staged by one CTA of 1024 threads per SM
        s->coarse_ok = s->coarse_on = s->split_ok_c = false;
        s->beam_smem_c = tab + (map->n_words + map->n_words_coarse) * sizeof(uint32_t);
        s->split_smem_c = step_split_smem_bytes(s->beam_smem_c, robot->V);
        s->beam_grid_c = s->split_grid_c = 0;
        const size_t cBitsR = coarse_words(map->H, map->dev.strideR) * 32, cBitsC = coarse_words(map->W, map->dev.strideC) * 32;
        if (e == cudaSuccess && s->use_smem && s->beam_smem_c <= (size_t)max_optin && cBitsR < (1u << 20) && cBitsC < (1u << 20)) {
            int f0 = 0, f1 = 0;
            e = kernel_config(beam_kernel<true, false, true>, 1024, s->beam_smem_c, max_optin, &f0);
            if (e == cudaSuccess && f0 >= 1) { s->coarse_ok = true; s->beam_grid_c = s->num_sms * f0; }
            if (e == cudaSuccess && s->coarse_ok && s->split_smem_c <= (size_t)max_optin) {
                e = kernel_config(step_beam_kernel<true, false, true>, 1024, s->split_smem_c, max_optin, &f1);
                if (e == cudaSuccess && f1 >= 1) { s->split_ok_c = true; s->split_grid_c = s->num_sms * f1; }
            }
            s->coarse_on = s->coarse_ok && kCoarseDefault;
        }
    }
    if (e != cudaSuccess) {
        int code = e == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA;
        fail(code, "fn_sim_create: %s", cudaGetErrorString(e));
        fn_sim_destroy(s);
        return code;
    }
    *out = s;
    return FN_OK;
}

extern "C" int fn_sim_destroy(fn_sim* s) {
    if (!s) return FN_OK;
    cudaFree(s->d_poses); cudaFree(s->d_ring_head); cudaFree(s->d_list); cudaFree(s->d_count); cudaFree(s->d_dprev);
    cudaFree(s->d_epstep); cudaFree(s->d_counters); cudaFree(s->d_task_counter);
    cudaFree(s->d_step_end);
    cudaFree(s->term.idx); cudaFree(s->term.id); cudaFree(s->term.start);
    cudaFree(s->d_prep.states); cudaFree(s->d_prep.goal_obs); cudaFree(s->d_prep.d_prev); cudaFree(s->d_prep.poses);
    cudaFree(s->d_prep.fail); cudaFree(s->d_prep_epstep);
    cudaFree(s->d_done_list); cudaFree(s->d_done_count); cudaFree(s->d_eval_outcome); cudaFree(s->d_eval_return);
    if (s->ev) { for (cudaEvent_t e : *s->ev) cudaEventDestroy(e); delete s->ev; delete s->ev_kind; }
    cudaFree(s->stg_states); cudaFree(s->stg_actions); cudaFree(s->stg_ranges); cudaFree(s->stg_gobs);
    cudaFree(s->stg_mask); cudaFree(s->stg_col); cudaFree(s->stg_seeds);
    if (s->pipe_init) {
        for (auto& h : s->hslot) {
            cudaFree(h.ranges); cudaFree(h.gobs); cudaFree(h.states); cudaFree(h.actions); cudaFree(h.mask); cudaFree(h.col); cudaFree(h.seeds);
            if (h.ev_ready) cudaEventDestroy(h.ev_ready);
            if (h.ev_done) cudaEventDestroy(h.ev_done);
        }
        if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
    }
    delete s;
    return FN_OK;
}

// Launch with the programmatic-stream-serialization attribute (PDL, fn_common.cuh).
template <class... KArgs, class... Args>
static cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

extern "C" int fn_sim_set_stream(fn_sim* s, void* stream) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_set_stream: NULL sim");
    s->stream = (cudaStream_t)stream;
    return FN_OK;
}

static int ring_row_floats(const fn_sim* s) { return s->robot->B + 5 + (s->robot->drive == FN_DRIVE_DIFF ? 2 : 3) + 2; }

// the launch for one sensor of the robot: its table, beam count, range, poses and block of the observation row
static BeamArgs beam_args(fn_sim* s, const int* list, const int* count_dev, float* out_ranges, bool step_launch, bool done_list,
                          int sensor = 0) {
    BeamArgs b;
    const fn_sensor& sn = s->robot->sensors[sensor];
    b.map = s->map->dev; b.robot = robot_dev(s->robot, s->map); b.poses = s->d_poses + (size_t)sensor * s->n; b.count_words = s->count_words;
    b.out_stride = (unsigned)s->robot->B; b.out_off = (unsigned)sn.off;
    b.robot.beam_cs += sn.off; b.robot.B = sn.B; b.robot.rmax = sn.rmax; b.robot.T = (double)sn.rmax / (double)s->map->res;
    b.list = list; b.count_dev = count_dev; b.n_all = s->n; b.out_ranges = out_ranges; b.out_hit = s->aux_hit;
    b.ring_obs = s->ring; b.ring_cap = s->ring_cap ? s->ring_cap : 1; b.ring_head = s->d_ring_head; b.ring_row = ring_row_floats(s);
    b.counters = s->d_counters; b.task_counter = s->d_task_counter;
    b.flip_par_dev = step_launch ? s->d_done_count + 2 : nullptr; b.done_count = s->d_done_count;
    b.list_par_dev = done_list ? s->d_done_count + 2 : nullptr;
    b.exp_off = kExpOff;
    b.pair_lines = b.robot.T >= 110.0;                             // beams of >~ 16 lines on average
    {   // ceil(2^32 / S) for S = bits per line (FastOrient::inv_magic)
        const unsigned long long SR = 32ull * (unsigned long long)s->map->dev.strideR, SC = 32ull * (unsigned long long)s->map->dev.strideC;
        b.inv_magicR = (unsigned)(((1ull << 32) + SR - 1) / SR); b.inv_magicC = (unsigned)(((1ull << 32) + SC - 1) / SC);
    }
    fast_chunking(sn.B, &b.chunk_rounds, &b.nchunk);
    {
        const unsigned long long rounds = ((unsigned long long)sn.B + 31) >> 5;
        b.inv_nchunk = fast_magic((unsigned long long)b.nchunk, (unsigned long long)s->n * b.nchunk);
        b.inv_rounds = fast_magic(rounds, (unsigned long long)s->n * rounds);
    }
    b.half_T = 0.5 * b.robot.T;
    return b;
}

// a sim sizes its poses, shared memory and output rows for the robot's sensors at fn_sim_create: every call
// that launches a kernel checks first that none was added since (the env kernels write one pose per sensor)
static int sensors_unchanged(const fn_sim* s) {
    if ((int)s->robot->sensors.size() != s->n_sensors)
        return fail(FN_ERR_INVALID_ARG, "the robot's sensors changed after fn_sim_create");
    return FN_OK;
}

static int launch_beams(fn_sim* s, const int* list, const int* count_dev, float* out_ranges, bool step_launch = false, bool done_list = false) {
    if (int rc0 = sensors_unchanged(s)) return rc0;
    const bool aux = s->count_words || s->aux_hit;
    const dim3 grid(s->beam_grid), block(kBeamThreads);
    for (int k = 0; k < s->n_sensors; ++k) {                      // one launch per sensor
        // (the kernel before the first launch has zeroed the dynamic task counter; the done-list parity flips once)
        if (k) FN_CUDA(cudaMemsetAsync(s->d_task_counter, 0, sizeof(unsigned), s->stream));
        const BeamArgs b = beam_args(s, list, count_dev, out_ranges, step_launch && k == 0, done_list, k);
        if (s->coarse_on && !aux) {
            FN_CUDA(launch_pdl(beam_kernel<true, false, true>, dim3(s->beam_grid_c), dim3(1024), s->beam_smem_c, s->stream, b));
        } else if (s->use_smem) {
            if (aux) FN_CUDA(launch_pdl(beam_kernel<true, true>, grid, block, s->beam_smem, s->stream, b));
            else FN_CUDA(launch_pdl(beam_kernel<true, false>, grid, block, s->beam_smem, s->stream, b));
        } else {
            if (aux) FN_CUDA(launch_pdl(beam_kernel<false, true>, grid, block, s->beam_smem, s->stream, b));
            else FN_CUDA(launch_pdl(beam_kernel<false, false>, grid, block, s->beam_smem, s->stream, b));
        }
    }
    return FN_OK;
}

// clearance features of all envs (list == NULL) or of the listed ones, from the ranges just written
static int launch_features(fn_sim* s, const int* list, const int* count_dev, bool done_list, const float* ranges) {
    if (!s->feat_z) return FN_OK;
    FeatArgs f;
    f.beam_cs = s->robot->d_beam_cs; f.verts = s->robot->d_verts; f.nxt = s->robot->d_nxt; f.B = s->robot->B; f.V = s->robot->V;
    f.n_sectors = s->feat_sectors; f.rmax = s->robot->rmax; f.sx = s->robot->sensor[0]; f.sy = s->robot->sensor[1];
    f.ranges = ranges; f.z = s->feat_z; f.list = list; f.count_dev = count_dev;
    f.list_par_dev = done_list ? s->d_done_count + 2 : nullptr; f.n_all = s->n;
    int grid = (s->n + kFeatEnvs - 1) / kFeatEnvs;
    if (grid > s->num_sms * 8) grid = s->num_sms * 8;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (s->prof) {
        FN_CUDA(cudaEventCreate(&e0)); FN_CUDA(cudaEventCreate(&e1));
        s->ev->push_back(e0); s->ev->push_back(e1); s->ev_kind->push_back(list ? 3 : 2);
        FN_CUDA(cudaEventRecord(e0, s->stream));
    }
    FN_CUDA(launch_pdl(features_kernel, dim3(grid), dim3(kFeatWarps * 32), feat_smem_bytes(f.V, f.n_sectors, f.B), s->stream, f));
    if (s->prof) FN_CUDA(cudaEventRecord(e1, s->stream));
    return FN_OK;
}

// evaluation is not training: between fn_eval_begin and fn_eval_end no call touches the replay ring, its
// head or the terminal observations
struct RingOff {
    fn_sim* s; float* keep;
    explicit RingOff(fn_sim* s_) : s(s_), keep(s_->ring) { if (s->eval_mode) s->ring = nullptr; }
    ~RingOff() { s->ring = keep; }
};

static ResetArgs reset_args(fn_sim* s, float* states, const int* list, const int* count, const int* list_par_dev,
                            const uint64_t* seeds, float* out_goal_obs) {
    ResetArgs a;
    a.map = s->map->dev; a.robot = robot_dev(s->robot, s->map); a.task = task_dev(s->task);
    a.regions.rects = s->map->d_regions; a.regions.n = s->map->n_regions;
    a.n = s->n; a.states = states; a.list = list; a.count_dev = count;
    a.list_par_dev = list_par_dev;
    a.seeds = reinterpret_cast<const unsigned long long*>(seeds); a.out_goal_obs = out_goal_obs;
    a.d_prev = s->d_dprev; a.ep_step = s->d_epstep; a.poses = s->d_poses;
    a.ring = s->ring; a.ring_cap = s->ring_cap ? s->ring_cap : 1; a.ring_head_dev = s->d_ring_head; a.ring_row = ring_row_floats(s);
    a.counters = s->d_counters; a.beam_task_counter = s->d_task_counter;
    a.fail_out = nullptr;
    return a;
}

// PAPER.md:84 "only the corresponding environments are reset and their observations recomputed": the reset itself (a
// chain of dependent map reads per env, ~10 us) does not depend on the step, only on the seeds -- announced before
// fn_step, it runs on the step kernel's outcome warps for the envs they report done, under the beam casting.
extern "C" int fn_sim_prepare_reset(fn_sim* s, const uint64_t* seeds) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_prepare_reset: NULL sim");
    s->prep_next = nullptr;
    if (!seeds || !s->prep_ok) return FN_OK;                       // (a hint: fn_reset gives the same result without it)
    if (!s->d_prep.states) {
        const size_t n = (size_t)s->n;
        cudaError_t e = cudaMalloc(&s->d_prep.states, 8 * n * sizeof(float));
        if (e == cudaSuccess) e = cudaMalloc(&s->d_prep.goal_obs, 2 * n * sizeof(float));
        if (e == cudaSuccess) e = cudaMalloc(&s->d_prep.d_prev, n * sizeof(float));
        if (e == cudaSuccess) e = cudaMalloc(&s->d_prep.poses, n * sizeof(BeamPose));
        if (e == cudaSuccess) e = cudaMalloc(&s->d_prep.fail, n);
        if (e == cudaSuccess) e = cudaMalloc(&s->d_prep_epstep, n * sizeof(int));
        if (e != cudaSuccess) {
            cudaFree(s->d_prep.states); cudaFree(s->d_prep.goal_obs); cudaFree(s->d_prep.d_prev); cudaFree(s->d_prep.poses);
            cudaFree(s->d_prep.fail); cudaFree(s->d_prep_epstep);
            s->d_prep = PreparedReset{}; s->d_prep_epstep = nullptr;
            return fail(e == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA, "fn_sim_prepare_reset: %s", cudaGetErrorString(e));
        }
    }
    s->prep_next = seeds;
    return FN_OK;
}

extern "C" int fn_step(fn_sim* s, float* states, const float* actions, float dt, uint8_t* reset_mask,
                       float* out_ranges, uint8_t* out_collision, float* out_goal_obs) {
    if (!s || !states || !actions || !reset_mask || !out_ranges || !out_collision || !out_goal_obs)
        return fail(FN_ERR_INVALID_ARG, "fn_step: NULL argument");
    if (!std::isfinite(dt) || dt < 0.0f) return fail(FN_ERR_INVALID_ARG, "fn_step: dt must be finite and >= 0");
    if (int rc0 = sensors_unchanged(s)) return rc0;
    RingOff ring_off(s);
    EnvArgs a;
    a.map = s->map->dev; a.robot = robot_dev(s->robot, s->map); a.task = task_dev(s->task);
    a.n = s->n; a.dt = dt; a.states = states; a.actions = actions; a.reset_mask = reset_mask;
    a.out_collision = out_collision; a.out_goal_obs = out_goal_obs; a.out_reward = s->aux_reward;
    a.d_prev = s->d_dprev; a.ep_step = s->d_epstep; a.poses = s->d_poses;
    a.ring = s->ring; a.ring_cap = s->ring_cap ? s->ring_cap : 1; a.ring_head_dev = s->d_ring_head; a.ring_row = ring_row_floats(s);
    a.counters = s->d_counters; a.beam_task_counter = s->d_task_counter;
    a.done_list = s->d_done_list; a.done_count = s->d_done_count; a.par_dev = s->d_done_count + 2;
    a.eval_outcome = s->eval_mode ? s->d_eval_outcome : nullptr; a.eval_return = s->d_eval_return; a.eval_limit = s->eval_limit;
    cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr;
    if (s->prof) {
        FN_CUDA(cudaEventCreate(&e0)); FN_CUDA(cudaEventCreate(&e1)); FN_CUDA(cudaEventCreate(&e2));
        s->ev->push_back(e0); s->ev->push_back(e1); s->ev->push_back(e2); s->ev_kind->push_back(0);
        FN_CUDA(cudaEventRecord(e0, s->stream));
    }
    a.epw = s->n >= 32768 ? 32 : (s->n >= 8192 ? 16 : 8);
    int rc = FN_OK;
    // announced seeds serve this step only; they are used when the production split step runs (no instruments, no
    // coarse level, training mode) and dropped otherwise -- fn_reset does the whole reset then, with the same result
    const uint64_t* prep_seeds = s->prep_next;
    s->prep_next = s->prep_ready = nullptr;
    if (!(s->prep_ok && s->split_on && !s->eval_mode && !s->count_words && !s->aux_hit && !(s->coarse_on && s->split_ok_c)))
        prep_seeds = nullptr;
    if (s->split_on) {
        // motion kernel, then the beam kernel whose last warps run collision / goal / reward / done for the
        // envs their CTAs own and whose last CTA advances the ring and the done-list parity (fn_step_split.cuh)
        FN_CUDA(launch_pdl(env_motion_kernel, dim3((s->n + a.epw - 1) / a.epw), dim3(kEnvBlock), 0, s->stream, a, s->d_step_end));
        if (s->prof) FN_CUDA(cudaEventRecord(e1, s->stream));
        const BeamArgs b = beam_args(s, nullptr, nullptr, out_ranges, false, false);
        const int epc = (s->n + s->split_grid - 1) / s->split_grid;
        const bool aux = s->count_words || s->aux_hit;
        const dim3 grid(s->split_grid), block(kBeamThreads);
        const unsigned bs = (unsigned)s->beam_smem;
        if (s->coarse_on && s->split_ok_c && !aux) {
            const int epc_c = (s->n + s->split_grid_c - 1) / s->split_grid_c;
            FN_CUDA(launch_pdl(step_beam_kernel<true, false, true>, dim3(s->split_grid_c), dim3(1024), s->split_smem_c, s->stream, b, a,
                               s->d_step_end, epc_c, (unsigned)s->beam_smem_c, 0));
        } else if (s->use_smem) {
            if (aux) FN_CUDA(launch_pdl(step_beam_kernel<true, true>, grid, block, s->split_smem, s->stream, b, a, s->d_step_end, epc, bs, 0));
            else if (prep_seeds) {
                // the resets of the envs this step reports done, prepared under the beam casting (fn_sim_prepare_reset)
                ResetArgs ra = reset_args(s, s->d_prep.states, nullptr, nullptr, nullptr, prep_seeds, s->d_prep.goal_obs);
                ra.d_prev = s->d_prep.d_prev; ra.ep_step = s->d_prep_epstep; ra.poses = s->d_prep.poses; ra.ring = nullptr;
                ra.fail_out = s->d_prep.fail;
                FN_CUDA(launch_pdl(step_beam_kernel<true, false, false, true>, grid, block, s->split_smem, s->stream, b, a, s->d_step_end, epc, bs, ra));
                s->prep_ready = prep_seeds; s->prep_map_ver = s->map->version; s->prep_robot_ver = s->robot->version;
            } else FN_CUDA(launch_pdl(step_beam_kernel<true, false>, grid, block, s->split_smem, s->stream, b, a, s->d_step_end, epc, bs, 0));
        } else {
            if (aux) FN_CUDA(launch_pdl(step_beam_kernel<false, true>, grid, block, s->split_smem, s->stream, b, a, s->d_step_end, epc, bs, 0));
            else FN_CUDA(launch_pdl(step_beam_kernel<false, false>, grid, block, s->split_smem, s->stream, b, a, s->d_step_end, epc, bs, 0));
        }
    } else {
        FN_CUDA(launch_pdl(env_step_kernel, dim3((s->n + a.epw - 1) / a.epw), dim3(kEnvBlock), col_scratch_bytes(s->robot->V), s->stream, a));
        if (s->prof) FN_CUDA(cudaEventRecord(e1, s->stream));
        if (s->ring) {
            FN_CUDA(launch_pdl(ring_advance_kernel, dim3(1), dim3(1), 0, s->stream, s->d_ring_head, (unsigned long long)s->n, s->ring_cap));
        }
        rc = launch_beams(s, nullptr, nullptr, out_ranges, true);
    }
    if (s->prof && rc == FN_OK) FN_CUDA(cudaEventRecord(e2, s->stream));
    if (rc == FN_OK) rc = launch_features(s, nullptr, nullptr, false, out_ranges);
    s->done_avail = 1;
    return rc;
}

extern "C" int fn_reset(fn_sim* s, float* states, const uint8_t* mask, const uint64_t* seeds,
                        float* out_ranges, float* out_goal_obs) {
    if (!s || !states || !seeds || !out_ranges || !out_goal_obs)
        return fail(FN_ERR_INVALID_ARG, "fn_reset: NULL argument");
    if (int rc0 = sensors_unchanged(s)) return rc0;
    if (!mask && !s->done_avail)
        return fail(FN_ERR_INVALID_ARG, "fn_reset: mask_dev == NULL needs a preceding fn_step (its done list is used once)");
    RingOff ring_off(s);
    const int* list = mask ? s->d_list : s->d_done_list;
    const int* count = mask ? s->d_count : s->d_done_count;
    if (!mask) s->done_avail = 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr, e3 = nullptr;
    if (s->prof) {
        FN_CUDA(cudaEventCreate(&e0)); FN_CUDA(cudaEventCreate(&e1)); FN_CUDA(cudaEventCreate(&e2)); FN_CUDA(cudaEventCreate(&e3));
        s->ev->push_back(e0); s->ev->push_back(e1); s->ev->push_back(e2); s->ev->push_back(e3); s->ev_kind->push_back(1);
        FN_CUDA(cudaEventRecord(e0, s->stream));
    }
    if (mask) FN_CUDA(launch_pdl(compact_mask_kernel, dim3(1), dim3(1024), 0, s->stream, mask, s->n, s->d_list, s->d_count));
    if (s->prof) FN_CUDA(cudaEventRecord(e1, s->stream));
    if (s->ring && s->term.term) {
        // the observations the step left behind are kept as next observations before the reset replaces them
        TerminalSaveArgs ta;
        ta.ring = s->ring; ta.head = s->d_ring_head; ta.cap = s->ring_cap; ta.n_envs = s->n; ta.row = ring_row_floats(s);
        ta.obs = s->robot->B + 5; ta.list = list; ta.count_dev = count; ta.list_par_dev = mask ? nullptr : s->d_done_count + 2;
        ta.td = s->term;
        int tg = (s->n + 7) / 8;
        if (tg > s->num_sms * 8) tg = s->num_sms * 8;
        FN_CUDA(launch_pdl(terminal_save_kernel, dim3(tg), dim3(256), 0, s->stream, ta));
    }
    const ResetArgs a = reset_args(s, states, list, count, mask ? nullptr : s->d_done_count + 2, seeds, out_goal_obs);
    int rc = FN_OK;
    // a reset prepared by the preceding fn_step for exactly this call (same seeds, nothing changed since)?
    const bool prepared = !mask && s->prep_ready == seeds && s->prep_map_ver == s->map->version && s->prep_robot_ver == s->robot->version &&
                          !s->count_words && !s->aux_hit;
    s->prep_ready = nullptr;
    // A CTA of the fused kernel runs its resets on kFusedResetWarps warps and casts only its own envs' beams:
    // made for the few envs a step reports done (C2, ~190 of 4096: 2-4 us faster than the two kernels).  For
    // long lists the two throughput-oriented kernels win (C2: all 4096 envs 83 against 121 us, a quarter of
    // them 38 against 47 us), and a caller's mask is usually such a list (the first reset of all envs), so
    // the fused kernel serves fn_reset(mask = NULL) only -- unless forced (enable = 2, tests).
    const bool fused = s->fused_on && (!mask || s->fused_force);
    if (prepared) {
        // one launch: copies of the prepared states and the beams of the listed envs, every warp of the grid taking rounds
        BeamArgs b = beam_args(s, list, count, out_ranges, false, true);
        b.poses = s->d_prep.poses;
        FN_CUDA(launch_pdl(prepared_reset_kernel, dim3(s->prep_grid), dim3(kBeamThreads), s->beam_smem, s->stream, a, b, s->d_prep,
                           (const StepEnd*)s->d_step_end, (unsigned)s->split_grid, s->prep_spin));
        if (s->prof) { FN_CUDA(cudaEventRecord(e2, s->stream)); FN_CUDA(cudaEventRecord(e3, s->stream)); }
    } else if (fused) {
        // one launch: every CTA resets its share of the list from its shared copy of the map, then casts
        // the beams of those envs (fn_reset_beam.cuh)
        BeamArgs b = beam_args(s, list, count, out_ranges, false, mask == nullptr);
        const bool aux = s->count_words || s->aux_hit;
        if (aux) FN_CUDA(launch_pdl(reset_beam_kernel<true>, dim3(s->fused_grid), dim3(kFusedThreads), s->fused_smem, s->stream, a, b));
        else FN_CUDA(launch_pdl(reset_beam_kernel<false>, dim3(s->fused_grid), dim3(kFusedThreads), s->fused_smem, s->stream, a, b));
        if (s->prof) { FN_CUDA(cudaEventRecord(e2, s->stream)); FN_CUDA(cudaEventRecord(e3, s->stream)); }
    } else {
        int grid = (s->n + kResetWarps - 1) / kResetWarps;
        if (grid > s->num_sms * 4) grid = s->num_sms * 4;
        FN_CUDA(launch_pdl(reset_kernel, dim3(grid), dim3(kResetWarps * 32), kResetWarps * col_scratch_bytes(s->robot->V), s->stream, a));
        if (s->prof) FN_CUDA(cudaEventRecord(e2, s->stream));
        rc = launch_beams(s, list, count, out_ranges, false, mask == nullptr);
        if (s->prof && rc == FN_OK) FN_CUDA(cudaEventRecord(e3, s->stream));
    }
    if (rc == FN_OK) rc = launch_features(s, list, count, mask == nullptr, out_ranges);
    return rc;
}

extern "C" int fn_observe_all(fn_sim* s, const float* states, float* out_ranges, float* out_goal_obs) {
    if (!s || !states || !out_ranges) return fail(FN_ERR_INVALID_ARG, "fn_observe_all: NULL argument");
    if (int rc0 = sensors_unchanged(s)) return rc0;
    RingOff ring_off(s);
    PoseArgs a;
    a.map = s->map->dev; a.robot = robot_dev(s->robot, s->map); a.n = s->n; a.states = states;
    a.out_goal_obs = out_goal_obs; a.poses = s->d_poses; a.beam_task_counter = s->d_task_counter;
    pose_from_state_kernel<<<(s->n + 255) / 256, 256, 0, s->stream>>>(a);
    FN_CUDA(cudaGetLastError());
    float* ring = s->ring;           // a test hook: never touches the ring
    s->ring = nullptr;
    int st = launch_beams(s, nullptr, nullptr, out_ranges);
    s->ring = ring;
    if (st == FN_OK) st = launch_features(s, nullptr, nullptr, false, out_ranges);
    return st;
}

extern "C" int fn_ranges_fixed_step(fn_sim* s, const float* states, float delta_m, int blockwise, float* out_ranges) {
    if (!s || !states || !out_ranges) return fail(FN_ERR_INVALID_ARG, "fn_ranges_fixed_step: NULL argument");
    if (!(delta_m > 0.0f) || !std::isfinite(delta_m)) return fail(FN_ERR_INVALID_ARG, "fn_ranges_fixed_step: delta must be > 0");
    if (int rc0 = sensors_unchanged(s)) return rc0;              // (the pose kernel writes one pose per LIVE sensor)
    if (s->n_sensors != 1) return fail(FN_ERR_UNSUPPORTED, "fn_ranges_fixed_step: comparison query, single-sensor robots only");
    PoseArgs a;
    a.map = s->map->dev; a.robot = robot_dev(s->robot, s->map); a.n = s->n; a.states = states;
    a.out_goal_obs = nullptr; a.poses = s->d_poses; a.beam_task_counter = s->d_task_counter;
    pose_from_state_kernel<<<(s->n + 255) / 256, 256, 0, s->stream>>>(a);
    FN_CUDA(cudaGetLastError());
    FixedStepArgs f;
    f.map = s->map->dev; f.poses = s->d_poses; f.beam_cs = s->robot->d_beam_cs; f.n = s->n; f.B = s->robot->B;
    f.delta_cells = delta_m / s->map->res; f.n_samples = (int)std::ceil((double)s->robot->rmax / (double)delta_m);
    f.rmax = s->robot->rmax; f.rho = s->map->res; f.out_ranges = out_ranges;
    const unsigned total = (unsigned)s->n * (unsigned)s->robot->B;
    if (blockwise) fixed_step_kernel<true><<<(total + 255) / 256, 256, 0, s->stream>>>(f);
    else fixed_step_kernel<false><<<(total + 255) / 256, 256, 0, s->stream>>>(f);
    FN_CUDA(cudaGetLastError());
    return FN_OK;
}

// ------------------------------------------------------------------------------------------ evaluation mode
extern "C" int fn_eval_begin(fn_sim* s, float* states, int n_cases, int step_limit, float* out_ranges, float* out_goal_obs) {
    if (!s || !states || !out_ranges || !out_goal_obs) return fail(FN_ERR_INVALID_ARG, "fn_eval_begin: NULL argument");
    if (n_cases < 1 || n_cases > s->n) return fail(FN_ERR_INVALID_ARG, "fn_eval_begin: n_cases must be in 1..n_envs");
    if (int rc0 = sensors_unchanged(s)) return rc0;
    if (step_limit < 1) return fail(FN_ERR_INVALID_ARG, "fn_eval_begin: the evaluation step limit must be >= 1");
    EvalBeginArgs a;
    a.pose.map = s->map->dev; a.pose.robot = robot_dev(s->robot, s->map); a.pose.n = s->n; a.pose.states = states;
    a.pose.out_goal_obs = out_goal_obs; a.pose.poses = s->d_poses; a.pose.beam_task_counter = s->d_task_counter;
    a.states = states; a.d_prev = s->d_dprev; a.ep_step = s->d_epstep; a.outcome = s->d_eval_outcome; a.ret = s->d_eval_return;
    a.n_cases = n_cases;
    eval_begin_kernel<<<(s->n + 255) / 256, 256, 0, s->stream>>>(a);
    FN_CUDA(cudaGetLastError());
    s->eval_mode = 1; s->eval_limit = step_limit; s->done_avail = 0;
    s->prep_next = s->prep_ready = nullptr;
    float* ring = s->ring;           // evaluation never touches the replay ring
    s->ring = nullptr;
    int st = launch_beams(s, nullptr, nullptr, out_ranges);
    s->ring = ring;
    if (st == FN_OK) st = launch_features(s, nullptr, nullptr, false, out_ranges);
    return st;
}

extern "C" int fn_eval_result(fn_sim* s, uint8_t* outcome, int32_t* steps, float* ret, int* n_running) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_eval_result: NULL sim");
    if (!s->eval_mode) return fail(FN_ERR_INVALID_ARG, "fn_eval_result: not in evaluation mode (fn_eval_begin)");
    std::vector<uint8_t> tmp((size_t)s->n);
    FN_CUDA(cudaMemcpyAsync(tmp.data(), s->d_eval_outcome, (size_t)s->n, cudaMemcpyDeviceToHost, s->stream));
    if (steps) FN_CUDA(cudaMemcpyAsync(steps, s->d_epstep, (size_t)s->n * sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    if (ret) FN_CUDA(cudaMemcpyAsync(ret, s->d_eval_return, (size_t)s->n * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
    FN_CUDA(cudaStreamSynchronize(s->stream));
    int running = 0;
    for (int e = 0; e < s->n; ++e) running += tmp[e] == 0;
    if (outcome) std::memcpy(outcome, tmp.data(), (size_t)s->n);
    if (n_running) *n_running = running;
    return FN_OK;
}

extern "C" int fn_eval_end(fn_sim* s) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_eval_end: NULL sim");
    s->eval_mode = 0;
    return FN_OK;
}

extern "C" int fn_sim_bind_aux(fn_sim* s, int32_t* hit, float* reward) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_bind_aux: NULL sim");
    s->aux_hit = hit; s->aux_reward = reward;
    return FN_OK;
}

extern "C" int fn_sim_bind_features(fn_sim* s, int n_sectors, float* out_z) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_bind_features: NULL sim");
    if (out_z) if (int rc0 = sensors_unchanged(s)) return rc0;   // (B below is the live robot's row length)
    if (out_z && s->n_sensors != 1) return fail(FN_ERR_UNSUPPORTED, "fn_sim_bind_features: single-sensor robots only");
    if (out_z && (n_sectors < 1 || n_sectors > s->robot->B))
        return fail(FN_ERR_INVALID_ARG, "fn_sim_bind_features: n_sectors must be in 1..B");
    if (out_z && feat_smem_bytes(s->robot->V, n_sectors, s->robot->B) > 48 * 1024)
        return fail(FN_ERR_UNSUPPORTED, "fn_sim_bind_features: too many sectors for shared memory");
    s->feat_z = out_z; s->feat_sectors = out_z ? n_sectors : 0;
    return FN_OK;
}

extern "C" int fn_ring_attach(fn_sim* s, float* ring, uint64_t cap) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_ring_attach: NULL sim");
    // a step completes the rows [head, head + n) and starts the pending rows [head + n, head + 2 n): below 2 n they alias
    if (ring && cap < 2 * (uint64_t)s->n) return fail(FN_ERR_INVALID_ARG, "fn_ring_attach: capacity must be >= 2 * n_envs");
    s->ring = ring; s->ring_cap = ring ? cap : 0;
    FN_CUDA(cudaMemsetAsync(s->d_ring_head, 0, 4 * sizeof(unsigned long long), s->stream));
    // a new ring starts without terminal observations (their indices refer to the old one)
    cudaFree(s->term.idx); cudaFree(s->term.id); cudaFree(s->term.start);
    s->term = TerminalDev{};
    return FN_OK;
}

extern "C" int fn_ring_attach_terminal(fn_sim* s, float* term, uint64_t rows) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_ring_attach_terminal: NULL sim");
    if (term && !s->ring) return fail(FN_ERR_INVALID_ARG, "fn_ring_attach_terminal: attach the ring first");
    if (term && rows < (uint64_t)s->n) return fail(FN_ERR_INVALID_ARG, "fn_ring_attach_terminal: rows must be >= n_envs (one reset may keep that many)");
    FN_CUDA(cudaStreamSynchronize(s->stream));
    cudaFree(s->term.idx); cudaFree(s->term.id); cudaFree(s->term.start);
    s->term = TerminalDev{};
    if (!term) return FN_OK;
    cudaError_t e = cudaMalloc(&s->term.idx, s->ring_cap * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&s->term.id, rows * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&s->term.start, rows * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemsetAsync(s->term.idx, 0xff, s->ring_cap * sizeof(int), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->term.id, 0xff, rows * sizeof(unsigned long long), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->term.start, 0, rows * sizeof(unsigned long long), s->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->d_ring_head + 2, 0, 2 * sizeof(unsigned long long), s->stream);
    if (e != cudaSuccess) {
        cudaFree(s->term.idx); cudaFree(s->term.id); cudaFree(s->term.start);
        s->term = TerminalDev{};
        return fail(e == cudaErrorMemoryAllocation ? FN_ERR_OOM : FN_ERR_CUDA, "fn_ring_attach_terminal: %s", cudaGetErrorString(e));
    }
    s->term.term = term; s->term.t_cap = rows; s->term.head = s->d_ring_head + 2;
    return FN_OK;
}

extern "C" int fn_ring_sample(fn_sim* s, uint64_t seed, int n_samples, float* out_rows, float* out_next_obs) {
    if (!s || !out_rows) return fail(FN_ERR_INVALID_ARG, "fn_ring_sample: NULL argument");
    if (!s->ring) return fail(FN_ERR_INVALID_ARG, "fn_ring_sample: no ring attached");
    if (n_samples < 1) return fail(FN_ERR_INVALID_ARG, "fn_ring_sample: n_samples must be >= 1");
    SampleArgs a;
    a.ring = s->ring; a.head = s->d_ring_head; a.cap = s->ring_cap; a.seed = seed; a.n_envs = s->n;
    a.row = ring_row_floats(s); a.obs = s->robot->B + 5; a.n_samples = n_samples;
    a.out_rows = out_rows; a.out_next_obs = out_next_obs; a.td = s->term;
    int grid = (n_samples + 7) / 8;
    if (grid > s->num_sms * 64) grid = s->num_sms * 64;
    FN_CUDA(launch_pdl(ring_sample_kernel, dim3(grid), dim3(256), 0, s->stream, a));
    return FN_OK;
}

extern "C" int fn_get_counters(fn_sim* s, uint64_t* host_out) {
    if (!s || !host_out) return fail(FN_ERR_INVALID_ARG, "fn_get_counters: NULL argument");
    FN_CUDA(cudaMemcpyAsync(host_out, s->d_counters, kNCounters * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s->stream));
    FN_CUDA(cudaStreamSynchronize(s->stream));
    return FN_OK;
}

extern "C" int fn_sim_profile(fn_sim* s, int enable) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_profile: NULL sim");
    if (!s->ev) { s->ev = new std::vector<cudaEvent_t>(); s->ev_kind = new std::vector<int>(); }
    s->prof = enable != 0;
    return FN_OK;
}

extern "C" int fn_sim_profile_read(fn_sim* s, double* ms_out, uint64_t* launches_out) {
    if (!s || !ms_out || !launches_out) return fail(FN_ERR_INVALID_ARG, "fn_sim_profile_read: NULL argument");
    for (int k = 0; k < 8; ++k) { ms_out[k] = 0.0; launches_out[k] = 0; }
    if (!s->ev) return FN_OK;
    FN_CUDA(cudaStreamSynchronize(s->stream));
    size_t i = 0;
    for (int kind : *s->ev_kind) {
        float ms = 0.f;
        if (kind == 0) {
            FN_CUDA(cudaEventElapsedTime(&ms, (*s->ev)[i], (*s->ev)[i + 1])); ms_out[0] += ms; launches_out[0] += 1;
            FN_CUDA(cudaEventElapsedTime(&ms, (*s->ev)[i + 1], (*s->ev)[i + 2])); ms_out[1] += ms; launches_out[1] += 1;
            i += 3;
        } else if (kind >= 2) {                                    // features kernel: all envs (2) / listed envs (3)
            FN_CUDA(cudaEventElapsedTime(&ms, (*s->ev)[i], (*s->ev)[i + 1])); ms_out[3 + kind] += ms; launches_out[3 + kind] += 1;
            i += 2;
        } else {
            for (int k = 0; k < 3; ++k) {
                FN_CUDA(cudaEventElapsedTime(&ms, (*s->ev)[i + k], (*s->ev)[i + k + 1])); ms_out[2 + k] += ms; launches_out[2 + k] += 1;
            }
            i += 4;
        }
    }
    for (cudaEvent_t e : *s->ev) cudaEventDestroy(e);
    s->ev->clear(); s->ev_kind->clear();
    return FN_OK;
}

extern "C" int fn_sim_beam_config(const fn_sim* s, int* cfg) {
    if (!s || !cfg) return fail(FN_ERR_INVALID_ARG, "fn_sim_beam_config: NULL argument");
    cfg[0] = s->use_smem ? 1 : 0; cfg[1] = s->beam_grid; cfg[2] = kBeamThreads; cfg[3] = (int)s->beam_smem;
    cfg[4] = s->split_on ? 1 : 0; cfg[5] = s->fused_on ? 1 : 0;
    cfg[6] = s->coarse_on ? 1 : 0; cfg[7] = s->coarse_ok ? 1 : 0;
    if (s->coarse_on) { cfg[1] = s->beam_grid_c; cfg[2] = 1024; cfg[3] = (int)s->beam_smem_c; }
    return FN_OK;
}

extern "C" int fn_sim_set_coarse(fn_sim* s, int enable, int* active_out) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_set_coarse: NULL sim");
    s->coarse_on = enable != 0 && s->coarse_ok;
    if (active_out) *active_out = s->coarse_on ? 1 : 0;
    return FN_OK;
}

extern "C" int fn_sim_set_fused_reset(fn_sim* s, int enable, int* active_out) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_set_fused_reset: NULL sim");
    s->fused_on = enable != 0 && s->fused_ok;
    s->fused_force = enable == 2;
    if (active_out) *active_out = s->fused_on ? 1 : 0;
    return FN_OK;
}

extern "C" int fn_sim_set_split_step(fn_sim* s, int enable, int* active_out) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_set_split_step: NULL sim");
    s->split_on = enable != 0 && s->split_ok;
    if (active_out) *active_out = s->split_on ? 1 : 0;
    return FN_OK;
}

extern "C" int fn_sim_count_words(fn_sim* s, int enable) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_count_words: NULL sim");
    s->count_words = enable != 0;
    return FN_OK;
}

extern "C" int fn_sim_episode_state(fn_sim* s, float* d_prev, int32_t* ep_step) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_sim_episode_state: NULL sim");
    if (d_prev) FN_CUDA(cudaMemcpyAsync(d_prev, s->d_dprev, (size_t)s->n * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
    if (ep_step) FN_CUDA(cudaMemcpyAsync(ep_step, s->d_epstep, (size_t)s->n * sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    FN_CUDA(cudaStreamSynchronize(s->stream));
    return FN_OK;
}

// ------------------------------------------------------------------------------------------ host buffers
extern "C" int fn_step_host(fn_sim* s, float* states, const float* actions, float dt, uint8_t* mask,
                            const uint64_t* seeds, float* out_ranges, uint8_t* out_collision, float* out_goal_obs) {
    if (!s || !states || !actions || !mask || !out_ranges || !out_collision || !out_goal_obs)
        return fail(FN_ERR_INVALID_ARG, "fn_step_host: NULL argument");
    const size_t n = (size_t)s->n, B = (size_t)s->robot->B, A = s->robot->drive == FN_DRIVE_DIFF ? 2 : 3;
    // each staging buffer on its own: the pipelined entry points share stg_states (pipe_alloc) and allocate none of
    // the others, and an allocation that failed half way must be completed by the next call, not skipped
    if (!s->stg_states) FN_CUDA(cudaMalloc(&s->stg_states, 8 * n * sizeof(float)));
    if (!s->stg_actions) FN_CUDA(cudaMalloc(&s->stg_actions, n * A * sizeof(float)));
    if (!s->stg_ranges) FN_CUDA(cudaMalloc(&s->stg_ranges, n * B * sizeof(float)));
    if (!s->stg_gobs) FN_CUDA(cudaMalloc(&s->stg_gobs, 2 * n * sizeof(float)));
    if (!s->stg_mask) FN_CUDA(cudaMalloc(&s->stg_mask, n));
    if (!s->stg_col) FN_CUDA(cudaMalloc(&s->stg_col, n));
    if (!s->stg_seeds) FN_CUDA(cudaMalloc(&s->stg_seeds, n * sizeof(unsigned long long)));
    cudaStream_t st = s->stream;
    FN_CUDA(cudaMemcpyAsync(s->stg_states, states, 8 * n * sizeof(float), cudaMemcpyHostToDevice, st));
    FN_CUDA(cudaMemcpyAsync(s->stg_actions, actions, n * A * sizeof(float), cudaMemcpyHostToDevice, st));
    FN_CUDA(cudaMemcpyAsync(s->stg_mask, mask, n, cudaMemcpyHostToDevice, st));
    if (seeds) FN_CUDA(cudaMemcpyAsync(s->stg_seeds, seeds, n * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
    // Ranges are 4 B per beam, the bulk of the output (12 MB of 12.2 MB at C2).  When the caller's buffer is
    // pinned (mapped) host memory and nothing on the device reads the ranges back (no feature kernel), the
    // beam kernels store them straight into it: each warp task writes 128 contiguous bytes, the stores are
    // posted over PCIe while the kernel computes, and the final device-to-host copy disappears.
    float* dev_ranges = s->stg_ranges;
    bool direct = false;
    if (!s->feat_z && n * B * sizeof(float) <= ((size_t)64 << 20)) {   // (larger outputs: the copy engine does as well)
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, out_ranges) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer) {
            dev_ranges = static_cast<float*>(pa.devicePointer);
            direct = true;
        } else {
            (void)cudaGetLastError();                              // (pageable memory: not an error here)
        }
    }
    int rc = seeds ? fn_sim_prepare_reset(s, reinterpret_cast<const uint64_t*>(s->stg_seeds)) : FN_OK;   // (the reset below)
    if (rc == FN_OK) rc = fn_step(s, s->stg_states, s->stg_actions, dt, s->stg_mask, dev_ranges, s->stg_col, s->stg_gobs);
    if (rc != FN_OK) return rc;
    // the step's own (pre-reset) outputs go back first; the reset then overwrites the done rows
    FN_CUDA(cudaMemcpyAsync(out_collision, s->stg_col, n, cudaMemcpyDeviceToHost, st));
    FN_CUDA(cudaMemcpyAsync(mask, s->stg_mask, n, cudaMemcpyDeviceToHost, st));
    if (seeds) {
        rc = fn_reset(s, s->stg_states, nullptr, reinterpret_cast<const uint64_t*>(s->stg_seeds), dev_ranges, s->stg_gobs);
        if (rc != FN_OK) return rc;
    }
    FN_CUDA(cudaMemcpyAsync(states, s->stg_states, 8 * n * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (!direct) FN_CUDA(cudaMemcpyAsync(out_ranges, s->stg_ranges, n * B * sizeof(float), cudaMemcpyDeviceToHost, st));
    FN_CUDA(cudaMemcpyAsync(out_goal_obs, s->stg_gobs, 2 * n * sizeof(float), cudaMemcpyDeviceToHost, st));
    FN_CUDA(cudaStreamSynchronize(st));
    return FN_OK;
}

// ------------------------------------------------------------------------------------------ host buffers, pipelined
// fn_step_host serialises copy in -> step -> reset -> copy out -> sync: at C2 the 12 MB of ranges take ~2.5x the
// step's own time on PCIe.  Here the states stay on the device, every step writes into one of two slots of
// device staging, and a slot's outputs drain on a copy stream while the next step already computes.
static int pipe_alloc(fn_sim* s) {
    if (s->pipe_init) return FN_OK;
    const size_t n = (size_t)s->n, B = (size_t)s->robot->B, A = s->robot->drive == FN_DRIVE_DIFF ? 2 : 3;
    std::memset(s->hslot, 0, sizeof(s->hslot));
    s->pipe_init = true;                                           // (fn_sim_destroy frees whatever was allocated)
    FN_CUDA(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
    if (!s->stg_states) FN_CUDA(cudaMalloc(&s->stg_states, 8 * n * sizeof(float)));
    for (auto& h : s->hslot) {
        FN_CUDA(cudaMalloc(&h.ranges, n * B * sizeof(float)));
        FN_CUDA(cudaMalloc(&h.gobs, 2 * n * sizeof(float)));
        FN_CUDA(cudaMalloc(&h.states, 8 * n * sizeof(float)));
        FN_CUDA(cudaMalloc(&h.actions, n * A * sizeof(float)));
        FN_CUDA(cudaMalloc(&h.mask, n));
        FN_CUDA(cudaMalloc(&h.col, n));
        FN_CUDA(cudaMalloc(&h.seeds, n * sizeof(unsigned long long)));
        FN_CUDA(cudaEventCreateWithFlags(&h.ev_ready, cudaEventDisableTiming));
        FN_CUDA(cudaEventCreateWithFlags(&h.ev_done, cudaEventDisableTiming));
    }
    return FN_OK;
}

extern "C" int fn_step_host_begin(fn_sim* s, int slot, const float* states_in, const float* actions, float dt,
                                  uint8_t* mask, const uint64_t* seeds, float* out_states, float* out_ranges,
                                  uint8_t* out_collision, float* out_goal_obs) {
    if (!s || !actions || !mask || !out_states || !out_ranges || !out_collision || !out_goal_obs)
        return fail(FN_ERR_INVALID_ARG, "fn_step_host_begin: NULL argument");
    if (slot < 0 || slot > 1) return fail(FN_ERR_INVALID_ARG, "fn_step_host_begin: slot must be 0 or 1");
    int rc = pipe_alloc(s);
    if (rc != FN_OK) return rc;
    fn_sim::HostSlot& h = s->hslot[slot];
    if (h.busy) return fail(FN_ERR_INVALID_ARG, "fn_step_host_begin: slot still in flight (call fn_step_host_end first)");
    if (!states_in && !s->pipe_states) return fail(FN_ERR_INVALID_ARG, "fn_step_host_begin: the first call must pass the states");
    const size_t n = (size_t)s->n, B = (size_t)s->robot->B, A = s->robot->drive == FN_DRIVE_DIFF ? 2 : 3;
    cudaStream_t st = s->stream;
    if (states_in) FN_CUDA(cudaMemcpyAsync(s->stg_states, states_in, 8 * n * sizeof(float), cudaMemcpyHostToDevice, st));
    s->pipe_states = true;
    FN_CUDA(cudaMemcpyAsync(h.actions, actions, n * A * sizeof(float), cudaMemcpyHostToDevice, st));
    FN_CUDA(cudaMemcpyAsync(h.mask, mask, n, cudaMemcpyHostToDevice, st));
    if (seeds) FN_CUDA(cudaMemcpyAsync(h.seeds, seeds, n * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
    if (seeds) rc = fn_sim_prepare_reset(s, reinterpret_cast<const uint64_t*>(h.seeds));                   // (the reset below)
    if (rc == FN_OK) rc = fn_step(s, s->stg_states, h.actions, dt, h.mask, h.ranges, h.col, h.gobs);
    if (rc != FN_OK) return rc;
    if (seeds) {
        rc = fn_reset(s, s->stg_states, nullptr, reinterpret_cast<const uint64_t*>(h.seeds), h.ranges, h.gobs);
        if (rc != FN_OK) return rc;
    }
    // the next step changes the states in place: the slot keeps this step's copy for the drain
    FN_CUDA(cudaMemcpyAsync(h.states, s->stg_states, 8 * n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    FN_CUDA(cudaEventRecord(h.ev_ready, st));
    FN_CUDA(cudaStreamWaitEvent(s->copy_stream, h.ev_ready, 0));
    cudaStream_t cs = s->copy_stream;
    FN_CUDA(cudaMemcpyAsync(out_ranges, h.ranges, n * B * sizeof(float), cudaMemcpyDeviceToHost, cs));
    FN_CUDA(cudaMemcpyAsync(out_states, h.states, 8 * n * sizeof(float), cudaMemcpyDeviceToHost, cs));
    FN_CUDA(cudaMemcpyAsync(out_goal_obs, h.gobs, 2 * n * sizeof(float), cudaMemcpyDeviceToHost, cs));
    FN_CUDA(cudaMemcpyAsync(out_collision, h.col, n, cudaMemcpyDeviceToHost, cs));
    FN_CUDA(cudaMemcpyAsync(mask, h.mask, n, cudaMemcpyDeviceToHost, cs));
    FN_CUDA(cudaEventRecord(h.ev_done, cs));
    h.busy = true;
    return FN_OK;
}

extern "C" int fn_step_host_end(fn_sim* s, int slot) {
    if (!s) return fail(FN_ERR_INVALID_ARG, "fn_step_host_end: NULL sim");
    if (slot < 0 || slot > 1) return fail(FN_ERR_INVALID_ARG, "fn_step_host_end: slot must be 0 or 1");
    if (!s->pipe_init || !s->hslot[slot].busy) return fail(FN_ERR_INVALID_ARG, "fn_step_host_end: nothing in flight in this slot");
    FN_CUDA(cudaEventSynchronize(s->hslot[slot].ev_done));
    s->hslot[slot].busy = false;
    return FN_OK;
}


// ------------------------------------------------------------------------------------------ fn_observe_noalloc
// fn_observe_all for callers that must not allocate device memory (include/flashnav.h says who they are).  The two
// kernels are the ones fn_observe_all launches -- pose_from_state_kernel, then the production beam kernel -- and
// what a sim would hold for them between the two launches lives in ONE statically sized device array instead:
//   bytes [0, 64)    the beam kernel's counters (kNCounters x u64; only "rays cast" is touched here)
//   bytes [128, 132) the beam kernel's dynamic task counter
//   bytes [256, ...) the sensing poses, FN_NOALLOC_MAX_ENVS x BeamPose
// The array is part of the loaded module: every device that loads libflashnav.so carries it (~0.75 MiB) until the
// process exits, whether or not this entry point is ever called.
constexpr size_t kNoallocHead = 256;
constexpr size_t kNoallocBytes = kNoallocHead + (size_t)FN_NOALLOC_MAX_ENVS * sizeof(BeamPose);
static_assert(kNCounters * sizeof(unsigned long long) <= 128 && kNoallocHead % alignof(BeamPose) == 0, "scratch layout");
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];

// In host code `g_noalloc_scratch` is only a handle for the symbol, never a device address: the address on a given
// device comes from cudaGetSymbolAddress with that device current, and differs from device to device.
constexpr int kNoallocMaxDevices = 64;
struct NoallocDevice {
    unsigned char* scratch;          // device address of g_noalloc_scratch on this device, NULL = not set up yet
    int num_sms, max_optin;
};
static NoallocDevice g_noalloc_dev[kNoallocMaxDevices];
static std::mutex g_noalloc_mutex;

// once per device, with that device current (the caller holds g_noalloc_mutex)
static int noalloc_setup(int dev, NoallocDevice* d) {
    unsigned char* p = nullptr;
    FN_CUDA(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
    if (!p) return fail(FN_ERR_CUDA, "fn_observe_noalloc: cudaGetSymbolAddress returned no address");
    FN_CUDA(cudaDeviceGetAttribute(&d->num_sms, cudaDevAttrMultiProcessorCount, dev));
    FN_CUDA(cudaDeviceGetAttribute(&d->max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    // raise the beam kernels' dynamic shared-memory limit to the device's opt-in maximum (what fn_sim_create does
    // for the sims; a function attribute, no memory involved)
    int unused = 0;
    FN_CUDA((beam_config<true, false>(0, d->max_optin, &unused)));
    FN_CUDA((beam_config<true, true>(0, d->max_optin, &unused)));
    FN_CUDA((beam_config<false, false>(0, d->max_optin, &unused)));
    FN_CUDA((beam_config<false, true>(0, d->max_optin, &unused)));
    d->scratch = p;
    return FN_OK;
}

extern "C" int fn_observe_noalloc(const fn_map* map, const fn_robot* robot, int n, const float* states,
                                  float* out_ranges, float* out_goal_obs, void* stream) {
    if (!map || !robot || !states || !out_ranges) return fail(FN_ERR_INVALID_ARG, "fn_observe_noalloc: NULL argument");
    if (n <= 0) return fail(FN_ERR_INVALID_ARG, "fn_observe_noalloc: n_envs must be > 0");
    const int n_sensors = (int)robot->sensors.size();
    if ((long long)n * n_sensors > (long long)FN_NOALLOC_MAX_ENVS)
        return fail(FN_ERR_INVALID_ARG, "fn_observe_noalloc: n_envs x sensors = %lld is beyond the static scratch of "
                    "FN_NOALLOC_MAX_ENVS = %d poses (use fn_sim_create + fn_observe_all for larger batches)",
                    (long long)n * n_sensors, (int)FN_NOALLOC_MAX_ENVS);
    if ((long long)n * robot->B >= (1ll << 31)) return fail(FN_ERR_UNSUPPORTED, "fn_observe_noalloc: n_envs * B must be < 2^31");
    int dev = 0;
    FN_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoallocMaxDevices) return fail(FN_ERR_UNSUPPORTED, "fn_observe_noalloc: device ordinal %d not supported", dev);
    NoallocDevice d;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_dev[dev].scratch)
            if (int rc = noalloc_setup(dev, &g_noalloc_dev[dev])) return rc;
        d = g_noalloc_dev[dev];
    }
    // A sim on the host stack that owns nothing: the scratch pointers go into the static array, everything a caller
    // could bind (ring, hit cells, features, coarse level) stays off, so launch_beams picks the production kernel
    // fn_observe_all runs for a sim without instruments.
    fn_sim shell;
    std::memset(&shell, 0, sizeof(shell));
    shell.map = map; shell.robot = robot; shell.n = n; shell.stream = (cudaStream_t)stream;
    shell.num_sms = d.num_sms; shell.n_sensors = n_sensors;
    shell.d_counters = reinterpret_cast<unsigned long long*>(d.scratch);
    shell.d_task_counter = reinterpret_cast<unsigned*>(d.scratch + 128);
    shell.d_poses = reinterpret_cast<BeamPose*>(d.scratch + kNoallocHead);
    {   // the beam launch configuration, by the rule of fn_sim_create (map staged in shared memory where it fits)
        const size_t tab = (size_t)robot->B * sizeof(double2);
        const size_t with_map = tab + map->n_words * sizeof(uint32_t);
        const double Tc = (double)robot->rmax / (double)map->res;
        const int Smin = 32 * ((map->dev.strideR < map->dev.strideC) ? map->dev.strideR : map->dev.strideC);
        const size_t rowBits = (size_t)(map->H + 2 * kLineGuard) * map->dev.strideR * 32;
        const size_t colBits = (size_t)(map->W + 2 * kLineGuard) * map->dev.strideC * 32;
        shell.use_smem = with_map + 8192 <= (size_t)d.max_optin && Tc + 34.0 < 0.5 * (double)Smin &&
                         rowBits < (1u << 20) && colBits < (1u << 20);
        shell.beam_smem = shell.use_smem ? with_map : tab;
        if (shell.beam_smem > (size_t)d.max_optin)
            return fail(FN_ERR_UNSUPPORTED, "fn_observe_noalloc: beam table does not fit in shared memory (B too large)");
        int bps = 0, bps2 = 0;
        if (shell.use_smem) {
            FN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, beam_kernel<true, false>, kBeamThreads, shell.beam_smem));
            FN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps2, beam_kernel<true, true>, kBeamThreads, shell.beam_smem));
        } else {
            FN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, beam_kernel<false, false>, kBeamThreads, shell.beam_smem));
            FN_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps2, beam_kernel<false, true>, kBeamThreads, shell.beam_smem));
        }
        if (bps2 < bps) bps = bps2;
        if (bps < 1) bps = 1;
        shell.beam_grid = d.num_sms * bps;
    }
    // What must start from zero: the task counter (the pose kernel zeroes it, as for fn_observe_all).  The counters
    // only ever accumulate and nobody reads them; the poses of all n envs are rewritten before the beam kernel reads.
    PoseArgs a;
    a.map = map->dev; a.robot = robot_dev(robot, map); a.n = n; a.states = states;
    a.out_goal_obs = out_goal_obs; a.poses = shell.d_poses; a.beam_task_counter = shell.d_task_counter;
    pose_from_state_kernel<<<(n + 255) / 256, 256, 0, shell.stream>>>(a);
    FN_CUDA(cudaGetLastError());
    return launch_beams(&shell, nullptr, nullptr, out_ranges);
}

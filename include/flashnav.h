/*
 * flashnav.h -- C ABI of libflashnav: the batched navigation-simulator step of FlashNav
 * (arxiv/paper_2606_15846), hand-written CUDA for sm_100a.
 *
 * One environment batch shares one occupancy bitmap; per step the library clips the
 * commands and advances the planar pose for the robot's drive type, tests the (possibly
 * nonconvex) footprint polygon against the map (Eq. (2) :118-123), computes goal
 * distance/direction, reward and termination (Eq. (1)), casts the range
 * beams, and on reset recomputes observations only for the environments that
 * were reset.  DESIGN.md states the readings taken where the paper is silent.
 *
 * Conventions
 *  - status: 0 = FN_OK, < 0 = error; fn_last_error() returns a thread-local message for the last error.
 *  - `*_host` pointers are host memory, copied during the call (the caller may free them at once).
 *  - `*_dev` pointers are caller-owned device memory on the current CUDA device; the library never
 *    frees them and keeps them only where stated (fn_sim_bind_aux, fn_ring_attach).
 *  - all work is enqueued on the CUDA stream given to fn_sim_create; calls return after enqueue and
 *    never synchronise, except fn_get_counters and the *_host convenience entry points.
 *  - argument errors are detected on the host before any launch; per-element problems (non-finite
 *    action, reset attempts exhausted) never fault: they bump device counters (fn_get_counters).
 *  - map frame: origin at the outer corner of cell (row 0, col 0); x grows with column, y with row;
 *    cell (i, j) = [j rho, (j+1) rho) x [i rho, (i+1) rho); linear cell index = i*W + j; everything
 *    outside the map is occupied.
 *  - there is no CPU fallback: every entry point that computes fails with FN_ERR_CUDA without a device.
 */
#ifndef FLASHNAV_H_
#define FLASHNAV_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { FN_OK = 0, FN_ERR_INVALID_ARG = -1, FN_ERR_UNSUPPORTED = -2, FN_ERR_OOM = -3, FN_ERR_CUDA = -4 };
enum { FN_DRIVE_DIFF = 0, FN_DRIVE_OMNI = 1 };
enum { FN_MAX_VERTS = 64, FN_MAX_ATTEMPTS = 256 };
enum { FN_N_COUNTERS = 8 };   /* rays cast, map words loaded, envs reset, reset failures,
                                 non-finite actions, env steps, map windows outside the packed map seen by
                                 the instrumented beam kernel (a self-check: must stay 0), envs whose reset
                                 was prepared by the step before (fn_sim_prepare_reset; also counted as reset) */

typedef struct fn_map fn_map;
typedef struct fn_robot fn_robot;
typedef struct fn_sim fn_sim;

/* ---- map ("the environment batch shares an occupancy bitmap") -------------------
 * bitmap_host: [H*W] row-major bytes, != 0 occupied.  The library bit-packs it (1 bit per cell) twice:
 * row-packed (bits along columns) and column-packed (bits along rows), each with a frame of occupied
 * cells around it ("outside the map is occupied"), and uploads both.
 * Errors: NULL pointers, H/W <= 0 or > 32768, resolution not finite or <= 0 -> FN_ERR_INVALID_ARG. */
int fn_map_create(const uint8_t* bitmap_host, int H, int W, float resolution_m, fn_map** out);

/* Optional sub-maps (BASELINE.json config 5: tiles of an atlas).  rects_host: [n][4] = row0, col0, h, w.
 * Environment e belongs to region e % n; fn_reset samples its start and goal inside that rectangle.
 * Beams and collision always see the whole map.  n = 0 clears the regions. */
int fn_map_set_regions(fn_map* map, int n, const int32_t* rects_host);
int fn_map_destroy(fn_map* map);

/* ---- robot specification xi = (F, S, K, U) ----------------------------------------
 * footprint_xy_host: [V][2] ordered polygon vertices, body frame, metres, CW or CCW, 3 <= V <= FN_MAX_VERTS.
 * beam_angles_host:  [B] beam directions in the body frame, radians, B >= 1.
 * drive_type: FN_DRIVE_DIFF commands (v_x, w); FN_DRIVE_OMNI commands (v_x, v_y, w).
 * vel_limits_host:   [6] = vx_min, vx_max, vy_min, vy_max, w_min, w_max (min <= max). */
int fn_robot_create(const float* footprint_xy_host, int V, const float* beam_angles_host, int B,
                    float max_range_m, int drive_type, const float* vel_limits_host, fn_robot** out);
/* Footprints that are a UNION of polygons ("polygon(s)"; :129 "For a union of polygons, the minimum
 * distance over its components is used"): footprint_xy_host holds the polygons' vertex lists one after the
 * other, comp_sizes_host [C] their vertex counts (each >= 3, total <= FN_MAX_VERTS).  The polygons may overlap;
 * the robot collides iff any of them does, a point is inside the footprint iff it is inside any of them. */
int fn_robot_create_union(const float* footprint_xy_host, const int32_t* comp_sizes_host, int C,
                          const float* beam_angles_host, int B, float max_range_m, int drive_type,
                          const float* vel_limits_host, fn_robot** out);
/* sensor placement S in the body frame; default (0, 0, 0). */
int fn_robot_set_sensor(fn_robot* robot, float sx_m, float sy_m, float spsi_rad);
/* A further range sensor (PAPER.md:65 "S defines sensor placement and range-sensing parameters"; :125): its own beam
 * table beam_angles_host [B] (rad, sensor frame), maximum range and placement (s_x, s_y, s_psi) in the body frame.
 * The observation row of an env becomes the concatenation of the sensors' ranges in the order they were added
 * (row length = sum of the beam counts: every [N][B] buffer of this header is sized with that sum); hit cells and
 * ring rows follow.  At most 4 sensors; call before fn_sim_create.  Each sensor is cast by its own beam launch
 * (fn_step / fn_reset then use the unfused launch sequences); clearance features and the fixed-step comparison
 * query are single-sensor (FN_ERR_UNSUPPORTED otherwise).  Errors: FN_ERR_INVALID_ARG, FN_ERR_UNSUPPORTED, FN_ERR_OOM. */
int fn_robot_add_sensor(fn_robot* robot, const float* beam_angles_host, int B, float max_range_m,
                        float s_x, float s_y, float s_psi);
/* acceleration limits of U: acc_host [3] = maximum |dv_x/dt|, |dv_y/dt|, |dw/dt| (> 0; +inf = none,
 * the default).  The clipped command is limited to the previous applied velocity (state planes 3..5)
 * +- a_max dt before the motion update.  Takes effect for sims created afterwards AND existing ones. */
int fn_robot_set_acc_limits(fn_robot* robot, const float* acc_host);
int fn_robot_destroy(fn_robot* robot);

/* ---- task parameters (Eq. (1); defaults via fn_task_default) ---------------------- */
typedef struct {
    float goal_tol_m;          /* goal reached when d < goal_tol_m           (default 0.3) */
    int   max_episode_steps;   /* 0 = no step limit                           (default 0)   */
    float goal_dist_min_m;     /* reset: goal distance range                  (default 3)   */
    float goal_dist_max_m;     /*                                             (default 8)   */
    float r_success;           /* Eq. (1)                                     (default 10)  */
    float r_collision;         /*                                             (default -10) */
    float c_progress;          /* c_1                                         (default 2)   */
} fn_task;
void fn_task_default(fn_task* out);

/* ---- simulator instance: n_envs environments on one map with one robot specification ----------------
 * cuda_stream: a cudaStream_t (NULL = the default stream).  The map and robot must outlive the sim. */
int fn_sim_create(const fn_map* map, const fn_robot* robot, int n_envs, const fn_task* task,
                  void* cuda_stream, fn_sim** out);
int fn_sim_destroy(fn_sim* sim);
/* Re-targets all later work of the sim to another stream (e.g. a capturing stream: fn_step / fn_reset only
 * enqueue kernels, never synchronise and keep all per-step state on the device, so a captured sequence of
 * them can be replayed as a CUDA graph).  The caller orders the old and the new stream. */
int fn_sim_set_stream(fn_sim* sim, void* cuda_stream);

/* ---- one vector step -------------------------------------------------------------------
 * states_dev:     [8][N] fp32 SoA planes x, y, psi, v_x, v_y, w, g_x, g_y; read and overwritten.
 * actions_dev:    [N][A] fp32, A = 2 (v_x, w) or 3 (v_x, v_y, w); clipped to the limits.
 * reset_mask_dev: [N] u8; in: forced-reset request, out: done = collision | goal reached | step limit | forced.
 * out_ranges_dev: [N][B] fp32 metres; out_collision_dev: [N] u8; out_goal_obs_dev: [2][N] fp32 (d, alpha).
 * Outputs are the PRE-reset observations ("Observations before reset are retained as next
 * observations in replay").  Call fn_reset with the done mask afterwards. */
int fn_step(fn_sim* sim, float* states_dev, const float* actions_dev, float dt, uint8_t* reset_mask_dev,
            float* out_ranges_dev, uint8_t* out_collision_dev, float* out_goal_obs_dev);

/* ---- reset of masked environments + selective observation recompute --------------
 * mask_dev: [N] u8, or NULL = exactly the envs the preceding fn_step reported done (their list is kept on the
 * device by fn_step, so no mask scan is needed; usable once per fn_step, else FN_ERR_INVALID_ARG);
 * seeds_dev: [N] u64 (one seed per env, read for masked envs only).
 * Rewrites ONLY the masked envs' state planes and their rows of out_ranges_dev / out_goal_obs_dev. */
int fn_reset(fn_sim* sim, float* states_dev, const uint8_t* mask_dev, const uint64_t* seeds_dev,
             float* out_ranges_dev, float* out_goal_obs_dev);

/* ---- optional outputs and hooks ---------------------------------------------------------------------------
 * fn_sim_bind_aux: extra per-step outputs, retained until re-bound or destroy; either may be NULL.
 *   out_hit_cell_dev [N][B] i32: linear cell index of the hit, -1 no hit, -2 outside the map.
 *   out_reward_dev   [N] fp32: Eq. (1).
 * fn_ring_attach: device replay ring (config 5).  Row = [ranges(B), d, alpha, v_x, v_y, w,
 *   action(A), reward, done] fp32; fn_step appends one row per env at slot (head + e) mod capacity, with
 *   obs = the observation the action was chosen from (the previous fn_step / fn_reset outputs).  done is a code:
 *   0 = the episode goes on, 1 = terminated (collision or goal reached), 2 = truncated (step limit or forced
 *   reset without a terminal event) -- the next observation of a done row is the post-reset one, so rows with
 *   code 2 cannot be bootstrapped from and a learner should leave them out or mask them.  A step
 *   completes the rows [head, head + N) and starts the next N, so capacity >= 2 N (else FN_ERR_INVALID_ARG).
 *   Evaluation steps (fn_eval_begin .. fn_eval_end) leave the ring and its head untouched.
 * fn_ring_attach_terminal: terminal observations ("Observations before reset are retained as next
 *   observations in replay, while reset observations are returned to the collector").  term_dev [rows][B + 5] fp32
 *   (the caller's, rows >= N) is a second ring: every fn_reset first copies, for each env it resets whose last
 *   completed ring row has a done code != 0, the observation the step left in the env's pending row -- [ranges(B),
 *   d, alpha, v_x, v_y, w], the pre-reset observation -- into the next entry (entries are reused in order), and
 *   fn_ring_sample returns it as the next observation of that row for as long as the entry exists.  Attach after
 *   fn_ring_attach (which drops it); NULL detaches.  Evaluation steps do not touch it.
 *   Errors: FN_ERR_INVALID_ARG (no ring, rows < N), FN_ERR_OOM / FN_ERR_CUDA (4 B per ring row + 8 B per entry).
 * fn_observe_all: recompute ranges and goal obs of ALL envs from states ("Full batch").
 * fn_get_counters: synchronises the stream and copies FN_N_COUNTERS u64 counters to host_out.
 * fn_sim_count_words: 1 = also count 32-bit map words loaded by the beam kernel (slower; default 0). */
int fn_sim_bind_aux(fn_sim* sim, int32_t* out_hit_cell_dev, float* out_reward_dev);
/* ---- clearance features (Eq. (3)): the policy's obstacle features z_t.
 * Each valid range endpoint (range < max range) is expressed in the body frame using the sensor placement;
 * delta_j = its distance to the footprint polygon (0 inside), capped at the max range; beams without a
 * valid hit get the max range; z_k = min of delta_j over sector k = the beams j with floor(j n_sectors / B) = k
 * (n_sectors groups of consecutive beams in table order; 1 <= n_sectors <= B).
 * out_z_dev [N][n_sectors] fp32 is retained until re-bound or destroy (NULL unbinds).  When bound, fn_step
 * writes the rows of all envs (from its pre-reset ranges), fn_reset rewrites the rows of the reset envs,
 * fn_observe_all writes all rows. */
int fn_sim_bind_features(fn_sim* sim, int n_sectors, float* out_z_dev);
int fn_ring_attach(fn_sim* sim, float* ring_dev, uint64_t capacity_transitions);
int fn_ring_attach_terminal(fn_sim* sim, float* term_dev, uint64_t rows);
/* ---- uniform replay sampling ("Each replay batch contains U x B transitions sampled uniformly
 * from replay and divided into U minibatches of size B"): gathers n_samples = U * B ring rows.
 * Sample i draws s = floor(SplitMix64(seed, i) * valid / 2^64), valid = min(rows completed, capacity - n_envs), and
 * takes slot (head - valid + s) mod capacity: uniform (with replacement) over the completed rows outside the
 * n_envs PENDING rows [head, head + n_envs), which already hold the next observation but stale action / reward /
 * done; nothing is written while no row is complete.
 * out_rows_dev [n_samples][B + 5 + A + 2] fp32: rows as stored (obs, action, reward, done) except for the done
 * code of truncated rows, see below;
 * out_next_obs_dev [n_samples][B + 5] or NULL: the obs part of the same env's next row (slot + n_envs mod
 * capacity), which the step that completed the row has already written -- for a done row the post-reset
 * observation, unless its terminal observation is kept (fn_ring_attach_terminal): then that one.  The done code of
 * the SAMPLED copy tells a learner what it got: 0 running, 1 terminated (bootstrap masked), 2 truncated with the
 * true pre-reset observation as next observation, 3 truncated but that observation is gone (entry reused, or no
 * terminal ring attached): not to be bootstrapped from.
 * Enqueued on the sim's stream, i.e. after the ring writes of earlier fn_step / fn_reset calls ("sampling waits
 * for the required replay writes"); the paper's two preallocated batch buffers are the caller's: alternate the
 * output pointers between calls and order the learner after the call with a stream or an event. */
int fn_ring_sample(fn_sim* sim, uint64_t seed, int n_samples, float* out_rows_dev, float* out_next_obs_dev);
int fn_observe_all(fn_sim* sim, const float* states_dev, float* out_ranges_dev, float* out_goal_obs_dev);
int fn_get_counters(fn_sim* sim, uint64_t* host_out);
int fn_sim_count_words(fn_sim* sim, int enable);
/* episode state kept by the sim, copied to HOST arrays d_prev_host [N] fp32 and ep_step_host [N] i32
 * (either may be NULL); synchronises the stream. */
int fn_sim_episode_state(fn_sim* sim, float* d_prev_host, int32_t* ep_step_host);

/* ---- live kernel timing (bench.py's roofline): when enabled, fn_step / fn_reset record CUDA events on
 * the sim's stream around their kernels.  fn_sim_profile_read synchronises, adds up the elapsed times
 * since the last read and clears them.  ms_out[8] / launches_out[8] = {env-step kernel, beam kernel of
 * fn_step, compaction kernel, reset kernel, beam kernel of fn_reset (the listed envs), features kernel of fn_step, features kernel of fn_reset, reserved}.
 * Events between kernels keep a kernel from starting under its predecessor (programmatic dependent
 * launch), so a profiled step is a few microseconds slower than an unprofiled one. */
int fn_sim_profile(fn_sim* sim, int enable);
int fn_sim_profile_read(fn_sim* sim, double* ms_out, uint64_t* launches_out);

/* ---- parallel policy evaluation: "Each batch assigns fixed start-goal cases to separate
 * environments ... Completion masks record each case once and exclude completed cases from further
 * accumulation of rewards and outcome statistics.  Each case ends when the robot reaches the goal, collides
 * with an obstacle, or reaches the evaluation step limit."
 * fn_eval_begin: states_dev [8][N] holds the start poses (planes 0-2) and goals (planes 6, 7) of the first
 *   n_cases envs (slots >= n_cases are inactive); zeroes the velocities, re-seeds the episode state, clears the
 *   completion masks, writes the initial observations of all envs and switches the sim to evaluation mode:
 *   fn_step then freezes every completed case (state and observation rows unchanged, reward 0, done 0 after
 *   the step that ended it), uses step_limit instead of the task's episode limit and does not need fn_reset.
 * fn_eval_result (synchronises): HOST arrays [N], any may be NULL: outcome u8 (0 running, 1 success, 2 collision,
 *   3 step limit, 4 inactive slot), steps i32 (steps taken; final for completed cases), return fp32 (sum of Eq. (1)
 *   rewards up to completion); *n_running = cases still running (0 = the batch has ended).
 * fn_eval_end: back to training mode (call fn_reset for all envs before stepping again). */
int fn_eval_begin(fn_sim* sim, float* states_dev, int n_cases, int step_limit, float* out_ranges_dev, float* out_goal_obs_dev);
int fn_eval_result(fn_sim* sim, uint8_t* outcome_host, int32_t* steps_host, float* return_host, int* n_running);
int fn_eval_end(fn_sim* sim);

/* ---- fn_observe_all without any allocation: ranges and goal observations of n_envs poses, no fn_sim -----------
 * For code that may not allocate device memory where it calls us.  Two kinds of caller are meant: (1) a process in
 * which a framework's pool (PyTorch's or JAX's allocator, an inference server) has already claimed all device
 * memory, so that a cudaMalloc from a third-party library fails or has to be routed through that pool; (2) a
 * control or serving loop with a latency bound, where cudaMalloc / cudaFree are ruled out because they synchronise
 * the whole device and stall every other stream.  fn_sim_create allocates per-sim buffers (poses, lists, counters);
 * this entry point needs no sim.  Its only working memory -- one sensing pose per env and sensor, between its two
 * kernels, plus the beam kernel's task and ray counters -- is a fixed array compiled into the library
 * (FN_NOALLOC_MAX_ENVS poses of 96 bytes + 256 bytes, about 0.75 MiB).  That array exists on every device that
 * loads the library, from load until the process exits, used or not.  The call makes no cudaMalloc, cudaFree or
 * other allocating call; it enqueues the same two kernels as fn_observe_all ("Full batch") on
 * cuda_stream and returns without synchronising, and its outputs are bit-identical to fn_observe_all's.
 *   map, robot:       handles made earlier, where allocating was still allowed (fn_map_create / fn_robot_create
 *                     upload the packed map and the tables); read only.  The robot's sensors all count:
 *                     n_envs x sensors <= FN_NOALLOC_MAX_ENVS.
 *   states_dev:       [8][N] fp32 planes as for fn_step (x, y, psi and the goal g_x, g_y are read).
 *   out_ranges_dev:   [N][B] fp32; out_goal_obs_dev: [2][N] fp32 or NULL.  All three are the caller's device memory.
 * First call on each device: looks up the array's address on that device (cudaGetSymbolAddress) and raises the
 * beam kernels' shared-memory limit, once, under a lock.  Make that first call at start-up, on the device it is
 * for and BEFORE any stream capture begins; later calls only launch.
 * Shared state: every call on a device uses the same array, whatever map, robot or stream it is given, and the
 * array keeps what the last call left (the task counter is cleared by the first kernel of each call, the poses are
 * rewritten before they are read, the ray counter just runs on).  Two calls that can overlap on the GPU -- different
 * streams without an event between them, or two host threads -- overwrite each other's poses: order them.
 * Errors: FN_ERR_INVALID_ARG (NULL argument, n_envs <= 0, n_envs x sensors > FN_NOALLOC_MAX_ENVS: the message says
 * so and names fn_sim_create + fn_observe_all as the way for larger batches), FN_ERR_UNSUPPORTED (beam table larger
 * than shared memory, n_envs x B >= 2^31), FN_ERR_CUDA. */
enum { FN_NOALLOC_MAX_ENVS = 8192 };
int fn_observe_noalloc(const fn_map* map, const fn_robot* robot, int n_envs, const float* states_dev,
                       float* out_ranges_dev, float* out_goal_obs_dev, void* cuda_stream);

/* ---- comparison only (not on the product path): the PAPER'S range query, "fixed-step samples along
 * each beam ... queried in distance blocks, and beams with a detected obstacle are removed from subsequent
 * blocks" (blockwise != 0), or its ablation baseline that evaluates all samples (blockwise == 0).
 * Sample k lies at k * delta_m from the sensor origin; range = distance of the first sample in an occupied
 * (or outside) cell, none below the max range => max range.  Writes out_ranges_dev [N][B] from states_dev;
 * both variants give the same ranges.  Overwrites the sim's sensing poses (like fn_observe_all). */
int fn_ranges_fixed_step(fn_sim* sim, const float* states_dev, float delta_m, int blockwise, float* out_ranges_dev);

/* ---- launch configuration chosen at fn_sim_create or by the switches below (for reports): cfg_out[8] =
 * {map staged in shared memory (1) or read through L1/L2 (0), beam grid size, CTA size, dynamic shared bytes,
 *  split step in use (fn_sim_set_split_step), fused reset in use for done lists (fn_sim_set_fused_reset),
 *  coarse level in use (fn_sim_set_coarse), coarse level available}. */
int fn_sim_beam_config(const fn_sim* sim, int* cfg_out);

/* ---- coarse level for empty-space skipping (BASELINE.json north_star).  Beside each packed copy
 * of the map the library keeps a coarse copy: one line per pair of lines, the OR of the two.  With enable != 0
 * the production beam kernels walk the coarse copy -- one 32-bit window per PAIR of lines -- and look at the two
 * fine lines only where that window is not empty; both variants resolve a hit on the same fine line with the
 * same fixed-point crossing coordinates, so ranges are bit-identical with the level on and off.  Available when
 * the map is staged in shared memory and fine + coarse copies fit one CTA (512 x 512 cells do).  *active_out (may
 * be NULL) = 1 if the level is available and enabled.  Host-side switch, takes effect at the next launch.
 * Errors: FN_ERR_INVALID_ARG (NULL sim). */
int fn_sim_set_coarse(fn_sim* sim, int enable, int* active_out);

/* ---- a reset announced before the step ("When episodes end, only the corresponding environments are
 * reset and their observations recomputed").  The reset of an env -- start pose and goal drawn from seeds[e] by the
 * rule of fn_reset -- does not depend on the step's result, only on WHICH envs end.  fn_sim_prepare_reset(sim,
 * seeds_dev) announces the seeds the fn_reset(mask = NULL) after the NEXT fn_step will be called with; that fn_step
 * then also runs the reset of every env it reports done, on the warps that compute the outcomes, into buffers of the
 * sim (states, outputs and the terminal observation of the step are what they are without the announcement), and the
 * fn_reset(sim, states, NULL, seeds_dev, ...) that follows copies those results and recomputes the observations.
 * Results are bit-identical with and without the announcement (tested).  The announcement serves one fn_step; it is
 * a hint and is dropped -- fn_reset then does the whole reset -- when the sim has no such kernel (map read through
 * L2, several sensors, instruments bound, coarse level, evaluation mode), when fn_reset is called with a mask or
 * other seeds, or when fn_map_set_regions / fn_robot_set_sensor ran in between.  seeds_dev = NULL withdraws an
 * announcement.
 * CONTRACT (not checkable by the library): seeds_dev [N] is READ DURING fn_step, and fn_reset recognises the
 * announcement by the ADDRESS of its seeds argument.  The buffer must hold the same values from fn_step until
 * fn_reset has been enqueued behind it; a buffer rewritten in place in between (one persistent seeds array refilled
 * every step) silently yields resets drawn from the values it held during fn_step, which then differ from the
 * un-announced path's (tests/test_gpu_parity.py pins this behaviour).  Refill before fn_sim_prepare_reset, or
 * alternate two buffers.
 * The fn_reset that applies a prepared reset starts under the tail of the preceding work in the stream, but writes
 * nothing of the caller's -- states, ranges, goal observations -- before that work has completed: a kernel the caller
 * enqueues between fn_step and fn_reset to read the pre-reset observation is safe, with or without programmatic
 * dependent launch.
 * Errors: FN_ERR_INVALID_ARG (NULL sim), FN_ERR_OOM / FN_ERR_CUDA (first call: the sim's buffers, 177 bytes per env). */
int fn_sim_prepare_reset(fn_sim* sim, const uint64_t* seeds_dev);

/* ---- fn_reset as one launch or two.  When the packed map is staged in shared memory (cfg_out[0] of
 * fn_sim_beam_config) and the reset scratch fits beside it, fn_reset(mask = NULL) -- the step's done list,
 * usually a few per cent of the envs -- runs ONE kernel in which every CTA resets its share of the listed envs
 * from its shared copy of the map and then recomputes their beams; this is the default
 * (enable = 1).  A caller's mask takes the two-kernel path (reset kernel, then the beam kernel over the list),
 * which is faster for long lists such as the first reset of all envs; enable = 0 uses it for the done list
 * too (worth it when a large part of the batch ends every step), enable = 2 uses the fused kernel for masks
 * as well (tests).  All paths give bit-identical states, goal observations and ranges.  *active_out (may be
 * NULL) = 1 if the fused kernel is available and enabled.  Host-side switch, takes effect at the next
 * fn_reset (a captured CUDA graph keeps the choice made at capture).  Errors: FN_ERR_INVALID_ARG (NULL sim). */
int fn_sim_set_fused_reset(fn_sim* sim, int enable, int* active_out);

/* ---- fn_step with the env step split around the beam kernel (default up to 64 envs per beam CTA, i.e. ~19 000
 * envs) or as one env-step kernel.  The beam
 * kernel needs only the new sensing poses, so by default fn_step launches a motion kernel (clip, motion update,
 * poses: PAPER.md:63) and a beam kernel in which the last warp of every CTA computes collision, goal
 * observation, reward and done for the envs the CTA owns while the other warps already cast
 * beams; the last CTA to finish advances the ring head and the done-list parity.  enable = 0 selects the
 * single env-step kernel followed by the ring-advance and beam kernels (also used when the collision scratch
 * does not fit beside the beam kernel's shared memory).  Both give bit-identical outputs.  *active_out (may
 * be NULL) = 1 if the split step will be used.  Host-side switch, takes effect at the next fn_step.
 * Errors: FN_ERR_INVALID_ARG (NULL sim). */
int fn_sim_set_split_step(fn_sim* sim, int enable, int* active_out);

/* ---- end-to-end convenience: host buffers in, host buffers out -----------------------------------------
 * Copies states/actions/mask (and seeds) host->device, runs fn_step (+ fn_reset of the done envs when
 * seeds_host != NULL), copies states, ranges, collision, goal obs and the done mask back, synchronises.
 * All pointers are HOST memory (pinned memory makes the copies asynchronous).  When out_ranges_host is pinned
 * (mapped) memory of at most 64 MB and no feature output is bound, the beam kernels store the ranges
 * straight into it over PCIe while they compute (no staging copy); the results are the same either way. */
int fn_step_host(fn_sim* sim, float* states_host, const float* actions_host, float dt,
                 uint8_t* reset_mask_host, const uint64_t* seeds_host, float* out_ranges_host,
                 uint8_t* out_collision_host, float* out_goal_obs_host);

/* ---- the same, pipelined over two slots: the copies of one step overlap the computation of the next.
 * fn_step_host_begin(slot) enqueues: host -> device of actions, forced-reset mask and seeds (and of the states when
 * states_in_host != NULL: the first call must pass them; NULL continues from the states the device holds), fn_step,
 * fn_reset of the done envs (when seeds_host != NULL), and -- on a copy stream, behind an event -- device -> host of
 * the post-reset states, the ranges (pre-reset rows of the envs that were not reset, post-reset rows of those that
 * were, like fn_step_host), the pre-reset collision flags, the goal observations and the done mask (written into
 * mask_host).  It returns after enqueueing.  fn_step_host_end(slot) blocks until that slot's outputs have arrived.
 * The next begin (other slot) may be issued before the end of this one: its kernels run while this slot drains
 * (at C2: 12 MB per step over PCIe against ~0.1 ms of computation).  Host buffers should be pinned and must stay
 * valid and untouched until the slot's end.  Errors: FN_ERR_INVALID_ARG (NULL, slot not 0 / 1, slot still in
 * flight, no states yet / nothing in flight), FN_ERR_OOM, FN_ERR_CUDA. */
int fn_step_host_begin(fn_sim* sim, int slot, const float* states_in_host, const float* actions_host, float dt,
                       uint8_t* mask_host, const uint64_t* seeds_host, float* out_states_host, float* out_ranges_host,
                       uint8_t* out_collision_host, float* out_goal_obs_host);
int fn_step_host_end(fn_sim* sim, int slot);

/* ---- roofline microbenchmarks (same binary, same run): bytes/s of conflict-free ld.shared.u32 x2
 * windows (kind 0), random-word ld.shared (kind 1) and L2-resident ld.global.nc (kind 2). */
int fn_measure_peak(int kind, void* cuda_stream, double* out_bytes_per_s);

const char* fn_last_error(void);
const char* fn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FLASHNAV_H_ */

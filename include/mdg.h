/* mdg.h — C ABI of the B200-native batched drone-environment step (libmdg.so).
 *
 * One call advances thousands of independent environments, each holding M Crazyflie-class quadrotors,
 * by one control step of arxiv/paper_2606_08039 ("MuJoCo-Drones-Gym"): action decode (PAPER.md:171-187
 * Table 3; cascaded PID PAPER.md:347-376), rotor model (Eq.1-3), ground effect / blade
 * drag / downwash (Eq.4-6), wind (Dryden-style gust, constant, impulse gusts,
 * sinusoidal), per-episode domain randomisation incl. motor lag, action / sensor latency and sensor noise (Table 4,
 * PAPER.md:229-248), free-body integration over
 * sim_freq/ctrl_freq substeps, observation, reward, termination and
 * auto-reset, and, as a separate call, the onboard depth / segmentation camera
 * (PAPER.md:177).  The interface follows the paper's statement of the
 * simulator: constructor options, `reset(rng) -> state`,
 * `step(state, action) -> state, obs, reward, done`.
 *
 * Conventions
 *  - Every function returns 0 (MDG_OK) or a negative error code; no exception or abort crosses the ABI.
 *    mdg_last_error() returns a thread-local description of the last failure.
 *  - "dev" pointers are CUDA device pointers on the device that was current at mdg_create; "host"
 *    pointers are ordinary host memory.  Library-owned buffers stay valid until mdg_destroy.
 *  - mdg_step / mdg_step_many / mdg_reset / mdg_gen_actions are asynchronous on the bound stream
 *    (default: the legacy default stream) and never synchronise.  mdg_get_* / mdg_set_* synchronise it.
 *  - A handle is not thread-safe; distinct handles are independent.
 *  - There is no CPU fallback: without a CUDA device mdg_create fails with MDG_ECUDA.
 */
#ifndef MDG_H
#define MDG_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define MDG_OK 0
#define MDG_EINVAL (-1) /* bad argument (n_envs<1, n_drones<1 or >32, unknown enum, sim_freq not a multiple of ctrl_freq) */
#define MDG_ECUDA (-2)  /* CUDA runtime error */
#define MDG_ENOMEM (-3) /* allocation failed */

/* aerodynamic feature mask ("toggled independently") */
enum { MDG_AERO_GND = 1, MDG_AERO_DRAG = 2, MDG_AERO_DW = 4, MDG_AERO_WIND = 8 };
enum { MDG_INTEG_RK4 = 0, MDG_INTEG_EULER = 1 };
enum { MDG_WIND_DRYDEN = 1, MDG_WIND_CONSTANT = 2, MDG_WIND_GUST = 4, MDG_WIND_SINE = 8 };   /* PAPER.md:199-205; all four = COMBINED */
/* Table 1 */
enum { MDG_PHYS_MJC = 0, MDG_PHYS_MJC_GND = 1, MDG_PHYS_MJC_DRAG = 2, MDG_PHYS_MJC_DW = 3,
       MDG_PHYS_MJC_GND_DRAG_DW = 4, MDG_PHYS_DYN = 5 };
/* Table 3.  Every action row is 4 floats per drone:
 *  RPM        raw rotor speeds, clipped to [0, MAX_RPM]
 *  PID        waypoint [x, y, z, psi] through the cascaded PID
 *  VEL        heading-frame [v_x, v_y, v_z, omega_z] through the same PID
 *  RPM_NORM   four rotor commands in [-1, 1] through normalizedActionToRPM: -1 -> 0, 0 -> HOVER_RPM,
 *             +1 -> MAX_RPM, piecewise linear, clipped (reading Q35)
 *  ONE_D_RPM  a[0] in [-1, 1] through the same map to all four rotors; a[1..3] ignored
 *  ATTITUDE   [thrust in [-1, 1] (same map, T = 4 k_f rpm^2), roll* rad, pitch* rad, yaw rate rad/s] through the
 *             attitude loop and the mixer of the cascaded PID (reading Q36) */
enum { MDG_ACT_RPM = 0, MDG_ACT_PID = 1, MDG_ACT_VEL = 2, MDG_ACT_RPM_NORM = 3, MDG_ACT_ONE_D_RPM = 4, MDG_ACT_ATTITUDE = 5 };
/* PAPER.md:177, 13.  KIN12 = [p, eta, v, omega]; KIN12_ADJ appends the adjacency row; KIN20 = [p, q, eta, v, omega,
 * a_{t-1}] with a_{t-1} the action applied in the step that produced the state (zeros after a reset). */
enum { MDG_OBS_KIN12 = 0, MDG_OBS_KIN12_ADJ = 1, MDG_OBS_KIN20 = 2, MDG_OBS_KIN12_TGT = 3 /* KIN12 + the 4 target words */,
       MDG_OBS_KIN12_WP = 4 /* KIN12 + next waypoint + its position in the body frame */,
       MDG_OBS_KIN12_Z = 5 /* KIN12 + the drone's target altitude: the 13-dim rows of MultiHoverAviary / MultiAgentAviary */ };
/* VELOCITY (VelocityAviary): target = (v*, omega_z*), r = -|v - v*| - 0.1 |omega_z - omega_z*| - 0.05 (|phi| + |theta|)
 * + 0.5 [|v - v*| < at_target_radius] summed over the env's drones */
enum { MDG_REW_HOVER = 0, MDG_REW_NEG_SQ_DIST = 1, MDG_REW_MULTI_HOVER = 2, MDG_REW_FORMATION = 3, MDG_REW_VELOCITY = 4,
       MDG_REW_FLY_THROUGH = 5 /* FlyThroughAviary: +10 per captured waypoint, -0.1 |d_wp|, -0.01 |omega|; the last capture terminates */ };
enum { MDG_TERM_NONE = 0, MDG_TERM_HOVER = 1, MDG_TERM_TILT_DIST = 2, MDG_TERM_FORMATION = 3 };
enum { MDG_LAYOUT_NONE = 0, MDG_LAYOUT_GRID = 1, MDG_LAYOUT_CIRCLE = 2 };
enum { MDG_TGT_FIXED = 0, MDG_TGT_SPAWN_LINSPACE = 1, MDG_TGT_BOX = 2, MDG_TGT_CIRCLE = 3,
       MDG_TGT_WAYPOINTS = 4 /* target = the waypoint being chased, 4th word = its index */ };
/* Table 2.  CF2P has CF2X's parameters and the +-configuration mixing:
 * tau_x = L (F_1 - F_3), tau_y = L (-F_0 + F_2) (reading Q37). */
enum { MDG_MODEL_CF2X = 0, MDG_MODEL_CF2P = 1, MDG_MODEL_RACE = 2 };

/* Plain-old-data parameter block.  struct_size must equal sizeof(mdg_params) (set by
 * mdg_default_params); units SI, rotor speeds in RPM, k_f and k_m per RPM^2 (DESIGN.md §3 Q1). */
typedef struct mdg_params {
    uint32_t struct_size;
    int32_t drone_model;
    /* Table 2 */
    float m, g, L, k_f, k_m, J[3], r_p, tw_ratio;
    /* Eq.4-6 coefficients; h_clip and dw_dz_clip regularise the h->0 and dz->0 singularities */
    float C_gnd, h_clip, c_xy, c_z, dw_C1, dw_C2, dw_C3, dw_dz_clip;
    /* wind gust: F = k_wind |w - v| (w - v); w <- a w + sigma sqrt(1-a^2) xi, a = exp(-dt_c/tau) */
    float k_wind, wind_sigma, wind_tau;
    int32_t sim_freq, ctrl_freq;   /* substeps per step = sim_freq / ctrl_freq */
    int32_t aero_mask, integrator; /* -1: derive from physics_mode (Table 1) */
    /* cascaded PID (Eq.9, Table 6) */
    float Kp_pos[3], Ki_pos[3], Kd_pos[3], Kp_att[3], Ki_att[3], Kd_att[3];
    float int_clamp_pos, int_clamp_att;
    int32_t dsl;                   /* 1: DSL-PID setpoint rate limits */
    float pos_rate_limit, yaw_rate_limit, a_ff[3], tilt_max, tau_xy_max, tau_z_max;
    /* observation, reward, termination */
    int32_t obs_mode; float adj_radius;
    int32_t reward_mode; float at_target_radius;
    int32_t term_mode; float term_tilt, term_dist, term_center[3], z_max;
    float episode_len_s; int32_t auto_reset;
    /* reset distribution and per-episode targets */
    int32_t reset_layout; float reset_center[3], reset_half[3], reset_z_lo, reset_z_hi;
    int32_t grid_cols; float grid_spacing, circle_radius;
    int32_t target_mode; float target_fixed[3], target_lo[3], target_hi[3], mh_z_lo, mh_z_hi,
        form_center[3], form_radius;
    /* global index of env 0: Philox counters use env_index_base + e, so a batch split across GPUs
     * draws exactly what the unsplit batch would (no collective on the step path) */
    uint32_t env_index_base;
    /* MDG_TGT_BOX: range of the 4th target word (VelocityAviary's yaw-rate target; 0, 0 by default) */
    float target_w_lo, target_w_hi;
    /* Domain randomisation (Table 4): half-widths a of the per-episode factors U(1-a, 1+a) applied to
     * [m, J, k_f, k_m, drag c_xy/c_z, C_gnd, downwash C_1, g, per-motor thrust bias (4 draws), arm L, MAX_RPM, -], redrawn at
     * every reset / auto-reset (vehicle factors per drone, g per env); all 0 = off.  The PID keeps the nominal model
     * (reading Q39).  reset_rpy_half / reset_vel_half: the table's initial-state ranges (uniform, 0 = at rest, level). */
    float dr_alpha[12];
    float reset_rpy_half[3], reset_vel_half[3];
    /* Table 4 motor lag (reading Q44): rotor speeds follow the command through a first-order lag, sampled exactly per
     * substep; the time constant is drawn per drone and episode from U(motor_lag_lo, motor_lag_hi) seconds (5-50 ms in the
     * table); 0, 0 = off.  Episodes start with the rotors at HOVER_RPM. */
    float motor_lag_lo, motor_lag_hi;
    /* Wind components (reading Q40), active when MDG_AERO_WIND is set: MDG_WIND_DRYDEN is the
     * AR(1) gust above (default), MDG_WIND_CONSTANT adds the steady air velocity wind_const (m/s) under the same quadratic
     * drag law, MDG_WIND_SINE adds the force wind_sine_amp [sin wt, cos wt, 0.3 sin 2wt] (N) of episode time t. */
    int32_t wind_mask; float wind_const[3], wind_sine_amp, wind_sine_omega;
    /* MDG_WIND_GUST (reading Q42): trigger probability per control step, largest impulse speed (m/s), impulse duration (s);
     * an impulse adds g sin(pi s) to the air velocity, direction uniform on the sphere, speed U(0, gust_max) */
    float gust_prob, gust_max, gust_duration;
    /* FlyThroughAviary: up to 8 ordered waypoints (x, y, z each) and the capture radius (reading Q41: 0.1 m) */
    int32_t n_waypoints; float waypoints[24], wp_radius;
    /* the waypoint-task family behind MDG_REW_FLY_THROUGH (reading Q43): reward per drone = wp_bonus [capture]
     * - wp_shaping |d_wp| + wp_speed |v| - wp_omega |omega|, the list run wp_laps times.  Defaults = FlyThroughAviary
     * (10, 0.1, 0, 0.01, 1 lap); RaceAviary = 20, 0.05, 2, 0, 2 laps over its six gates. */
    float wp_bonus, wp_shaping, wp_speed, wp_omega; int32_t wp_laps;
    /* Table 4 "sensors" rows and the sticky per-episode observation bias of PAPER.md:248 (iii) (DESIGN.md
     * reading Q49): standard deviations for [position m, velocity m/s, roll/pitch/yaw rad, body rates rad/s].  obs_noise is
     * drawn afresh for every emitted observation (Table 4: 0.01, 0.05, 1 degree = 0.01745, 0.05), obs_bias once per drone and
     * episode; both are Gaussian, added to the twelve kinematic entries of the MDG_OBS_* row only (quaternion, last action,
     * targets and adjacency stay exact); the simulated state, the controller, reward and termination see the true values.
     * All 0 (default) = off.  Negative values are MDG_EINVAL. */
    float obs_noise[4], obs_bias[4];
    /* MDG_WIND_DRYDEN with the altitude-dependent length scale (L_u = h / (0.177 + 8.23e-4 h)^1.2,
     * alpha = exp(-dt V / L); reading Q50): dryden_airspeed = V in m/s (0, the default, keeps the fixed wind_tau),
     * h = the mean altitude of the env's drones at the start of the control step, not below dryden_h_min (0.05 m). */
    float dryden_airspeed, dryden_h_min;
    /* Table 4 latency rows (reading Q51), ranges in seconds, one delay per drone and episode,
     * uniform over the whole numbers of physics substeps round(lo sim_freq) .. round(hi sim_freq); hi = 0 (default) = off.
     * Action latency (table: 0 - 0.050; at most 3 control steps): the row issued at a control step takes effect that many
     * substeps later; rotor-command rows (RPM, RPM_NORM, ONE_D_RPM) switch at the exact substep, the controller types decode
     * once per control step from the row that has arrived by then; until the episode's first row arrives that row is used.
     * Sensor latency (table: 0 - 0.020; at most 1 control step): the kinematic entries of the observation (p, quaternion,
     * roll/pitch/yaw, v, body rates) are the state that many substeps before the end of the step; the first row after a
     * reset / auto-reset is the initial state.  Both outside their window: MDG_EINVAL. */
    float act_latency_lo, act_latency_hi, obs_latency_lo, obs_latency_hi;
    /* FormationAviary's moving centre ("the formation centre tracks a closed polygonal path"; reading Q52),
     * with MDG_TGT_CIRCLE: form_path_n (2..8) vertices (x, y, z each) traversed at form_speed m/s from vertex 0 at episode time 0
     * and closed back to it; the circle slots (the per-drone targets, rewritten every step), the formation reward and the
     * distance rule of MDG_TERM_FORMATION follow the centre at the end-of-step time.  form_path_n < 2 or form_speed = 0
     * (default) = the static form_center / term_center. */
    int32_t form_path_n; float form_path[24], form_speed;
} mdg_params;

typedef struct mdg_env mdg_env; /* opaque; the library owns it and all its device buffers */

/* Fill *out (host pointer, caller-owned) with Table 2 of the drone model, the PIDControl gains of Table 6
 * (PAPER.md:365-372), the Eq.4-6 coefficients and the documented defaults of every other field.
 * MDG_EINVAL: NULL, unknown drone_model. */
int mdg_default_params(int drone_model, mdg_params* out);

/* Kernel selection: the five BASELINE configs and a few variants have precompiled instances of the step kernel; for any other
 * combination of modes and params mdg_create compiles an instance for exactly that combination with NVRTC (about a second, cached
 * per process; the sources are the csrc/ files beside the library) and falls back to a runtime-flag generic kernel if that is not
 * possible.  The fallback is 1.7-2.1x slower but not an error: mdg_create still returns MDG_OK, mdg_kernel_name says
 * "generic", and mdg_last_error() right after mdg_create holds the reason.  Environment variable MDG_JIT=0 forces the generic
 * kernel, MDG_JIT=require makes mdg_create fail with MDG_ECUDA instead of falling back; MDG_JIT_SRC overrides the directory
 * the sources are read from.
 *
 * Create n_envs environments of n_drones (1..32) drones each: the constructor of PAPER.md:169 (drone model, num_drones,
 * physics, sim / ctrl frequency, obs and act type) and, for the batch, MJXVectorAviary's num_envs.
 * physics_mode: Table 1; action_type: Table 3.  params (host, copied) may be NULL for the
 * CF2X defaults.  *out receives the handle; it owns all device memory (one arena) until mdg_destroy.  The state is that of
 * mdg_reset(env, 0).  Errors: MDG_EINVAL (see the code's comment above), MDG_ENOMEM, MDG_ECUDA (no device: no CPU fallback). */
int mdg_create(int n_envs, int n_drones, int physics_mode, int action_type, const mdg_params* params,
               mdg_env** out);
/* Free the handle and everything it owns (synchronises its stream).  NULL is ignored. */
void mdg_destroy(mdg_env* env);

/* The paper's `reset(rng) -> state` for the whole batch (per-env PRNG key, step counter and done flag of
 * MJXState): draw every env's initial state (Table 4's initial-state ranges when set) and
 * per-episode targets from Philox4x32-10 keyed by seed (counter = env_index_base + env, drone, 0, stream);
 * zero controller memory, wind and step counters; obs is valid afterwards (reward 0, done 0).  Asynchronous on the bound
 * stream.  MDG_EINVAL: NULL handle. */
int mdg_reset(mdg_env* env, uint64_t seed);

/* One control step: the paper's `step(state, action) -> state, obs, reward, done` for every env, i.e. action
 * decode (Table 3; PID PAPER.md:347-376), Eq.1-6 wrench, sim_freq/ctrl_freq integration
 * substeps, observation / reward / termination and same-call auto-reset
 * (PAPER.md:254-258), in one kernel launch.  actions_dev: [n_envs*n_drones][4] fp32, caller-owned device memory, 16-byte
 * aligned, read only; the meaning of the four floats follows the action type (see MDG_ACT_* above).  Asynchronous on the bound
 * stream, with plain stream semantics: the step starts after everything enqueued before it on that stream has completed
 * (so a policy kernel or mdg_gen_actions may write actions_dev right before it), and everything enqueued after
 * it sees its outputs complete.  MDG_EINVAL: NULL or misaligned argument. */
int mdg_step(mdg_env* env, const float* actions_dev);

/* The same step for callers whose actions do not come from the stream: the step is launched with programmatic dependent launch
 * and, when the previous operation on this handle was a step on the same stream, does NOT wait for the previous kernel of the
 * stream as a whole; it orders itself behind the previous step of this handle work item by work item, so the drain
 * of one step overlaps the ramp-up of the next, and steps of other handles enqueued in between overlap as well.
 * CONTRACT: the contents of actions_dev must have been complete and visible before the previous step of this handle was enqueued
 * (pre-generated action sets, buffers whose producer a full stream / event dependency ordered before that step).  With an
 * in-stream producer between two steps use mdg_step.  Everything enqueued after the step still sees it complete.  The first step
 * after any other operation on the handle (reset, set_state, load, render, set_stream, a graph replay) behaves like mdg_step.
 * The paper's counterpart is the jitted `lax.scan` of K sub-steps inside one call: work queued ahead, no host
 * round trip.  Same arguments and errors as mdg_step. */
int mdg_step_chained(mdg_env* env, const float* actions_dev);

/* n_steps control steps (each exactly mdg_step) replayed as one CUDA graph: step k reads actions_dev +
 * k*stride_floats; all n_steps action sets must be complete before the call.  Inside the graph the steps chain like
 * mdg_step_chained; the first waits for whatever precedes the replay.  The graph is cached per (pointer, n_steps, stride) and can
 * be replayed any number of times, between other steps; mdg_reset / mdg_load / mdg_set_launch drop the cache (seed and launch
 * shape are kernel parameters).  Outputs hold the last step's values.
 * MDG_EINVAL: NULL, n_steps < 1, misaligned pointer or stride. */
int mdg_step_many(mdg_env* env, const float* actions_dev, int n_steps, int64_t stride_floats);

/* One control step (exactly mdg_step) with HOST buffers, the end-to-end call a Gymnasium-style host loop
 * makes: copies actions_host [n_envs*n_drones][4] to
 * the device, steps, copies obs / reward / done back (NULL outputs are skipped) and synchronises the
 * stream, so the results are valid on return.  Pinned host memory makes the copies asynchronous
 * with respect to the host but the call still returns only after they finish.  obs_host [n_envs][mdg_obs_dim] fp32,
 * reward_host [n_envs] fp32, done_host [n_envs] u8; all caller-owned.  MDG_EINVAL: NULL handle or actions. */
int mdg_step_host(mdg_env* env, const float* actions_host, float* obs_host, float* reward_host, uint8_t* done_host);

/* The same call split in two, for double-buffering several handles (each bound to its own stream with mdg_set_stream) so that
 * one batch's device-to-host copy overlaps another batch's host-to-device copy and step: mdg_step_host_async enqueues the copy
 * of the actions, the step and the copies of the outputs on the bound stream and returns at once; the host buffers must be
 * pinned (page-locked) for the copies to be asynchronous and must not be touched until mdg_wait on the same handle has
 * returned.  mdg_wait blocks until everything enqueued on the handle's stream has finished.  mdg_step_host = async + wait. */
int mdg_step_host_async(mdg_env* env, const float* actions_host, float* obs_host, float* reward_host, uint8_t* done_host);
int mdg_wait(mdg_env* env);

/* mdg_step_host for callers that must not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same control step with the same arguments, results and
 * synchronisation as mdg_step_host, but the device staging buffer of the actions is a static device array inside the library
 * instead of a buffer mdg_step_host cudaMallocs on a handle's first call.  The call allocates and frees nothing, on the host
 * side of CUDA or the device.  Limits and caveats:
 *  - the array holds MDG_STATIC_STAGE_MAX_DRONES action rows (4 MiB; every GPU that loads the library holds it until the
 *    process exits); a handle with n_envs * n_drones beyond that gets MDG_EINVAL and a message naming both numbers;
 *  - there is ONE array per GPU, shared by every handle and thread of the process: calls that overlap on the GPU (two
 *    threads, each on its own handle and stream) race on it and step with mixed actions - serialise them, or use
 *    mdg_step_host, whose staging buffer is per handle.  The call itself returns only after its own work has finished;
 *  - the array keeps the previous call's rows; nothing in it has to start at zero, the call overwrites every row it reads.
 * Errors: MDG_EINVAL (NULL handle or actions, too many drones), MDG_ECUDA. */
#define MDG_STATIC_STAGE_MAX_DRONES 262144
int mdg_step_host_static(mdg_env* env, const float* actions_host, float* obs_host, float* reward_host, uint8_t* done_host);

/* Device pointers to the library-owned outputs of the last reset/step (`obs, reward, done` of PAPER.md:285-289; observation
 * rows PAPER.md:177, rewards and termination rules PAPER.md:304-333):
 * obs [n_envs][mdg_obs_dim] fp32 (per drone: the MDG_OBS_* row, e.g. p, roll/pitch/yaw, v, body rates [, adjacency row]);
 * reward [n_envs] fp32; done [n_envs] u8 (bit0 terminated, bit1 truncated).  Any may be NULL. */
int mdg_outputs(mdg_env* env, const float** obs_dev, const float** reward_dev, const uint8_t** done_dev);
int mdg_obs_dim(const mdg_env* env); /* floats per env = n_drones x the MDG_OBS_* row length; negative code on NULL */

/* Device pointer to the per-episode targets [n_envs*n_drones][4] = (x, y, z, psi), fp32: the task's hover point, velocity
 * target, waypoint or formation slot.  Library-owned, rewritten by reset / auto-reset (and every step for
 * waypoint and moving-formation tasks). */
int mdg_targets(mdg_env* env, const float** targets_dev);

/* Harness action generator, not part of the paper's method (it stands in for the policy of PAPER.md:285-292 so that tests and
 * bench.py can produce seeded actions on the device).  Philox stream 3, counter = (env_index_base + env, drone, t, 3):
 * out_dev[(e*n_drones+i)*4 + c] = base * fma(hi - lo, u_c, lo), every operation rounded to fp32.  out_dev: caller-owned
 * device memory, 16-byte aligned.  Asynchronous on the bound stream. */
int mdg_gen_actions(mdg_env* env, uint64_t seed, uint32_t t, float base, float lo, float hi, float* out_dev);

/* Checkpoint / test hooks (host pointers; synchronise the stream): the kinematic part of the paper's per-env state
 * (MJXState's qpos / qvel, step counter: PAPER.md:254-258; controller memory of PAPER.md:347-357).
 * state: [D][13] = p(3) q(4, w x y z) v(3) body rates(3);  ctrl: [D][10] = I_p(3) I_eta(3) held
 * setpoint(4);  targets: [D][4];  wind: [n_envs][3];  ep_step: [n_envs] u32.  D = n_envs*n_drones.
 * NULL pointers are skipped.  mdg_set_state recomputes obs. */
int mdg_get_state(mdg_env* env, float* state, float* ctrl, float* targets, float* wind, uint32_t* ep_step);
int mdg_set_state(mdg_env* env, const float* state, const float* ctrl, const float* targets,
                  const float* wind, const uint32_t* ep_step);

/* Full checkpoint / resume of everything MJXState carries (data, step counter, PRNG key, done) and this
 * library adds.  mdg_get_state covers the kinematic state for tests; a running simulation also carries the DR
 * factors, rotor speeds (motor lag), gust impulses, action history (action latency), step counters, the seed and the last
 * outputs.  mdg_save writes all of it to host memory as one opaque blob of mdg_checkpoint_size bytes; mdg_load restores it
 * into a handle created with the same n_envs, n_drones, modes and params, after which stepping continues bit for bit as
 * if never interrupted.  Both synchronise the stream.  MDG_EINVAL: NULL, short buffer, a blob of another library version or
 * of a handle with another shape / feature set.  mdg_checkpoint_size returns a negative code on a NULL handle. */
int64_t mdg_checkpoint_size(const mdg_env* env);
int mdg_save(mdg_env* env, void* host_buf, int64_t buf_bytes);
int mdg_load(mdg_env* env, const void* host_buf, int64_t buf_bytes);

/* Per-agent view for multi-agent training (MultiAgentAviary): device pointer to [n_envs*n_drones] fp32, each
 * drone's share of the last step's reward (its own terms plus half of every pair term it is part of); the shares of an
 * env add up to its reward.  Library-owned, valid until mdg_destroy; written by every mdg_step. */
int mdg_reward_per_drone(mdg_env* env, const float** reward_dev);

/* Domain-randomisation factors of the running episodes (Table 4), host [D][16] = [m, J, k_f, k_m, drag, C_gnd, C_1, g, motor bias x4,
 * arm, MAX_RPM, motor-lag time constant (s; 1 when off), 1] (synchronise).
 * mdg_set_dr fails with MDG_EINVAL when every dr_alpha is 0 (the factors are then not read by the step). */
int mdg_get_dr(mdg_env* env, float* factors);
int mdg_set_dr(mdg_env* env, const float* factors);

/* Onboard depth / segmentation camera (48 x 64 frames from each drone's 60-degree-FOV camera positioned at
 * [0.02, 0, 0] in the body frame; PAPER.md:13 lists RGB / depth / segmentation).  The paper renders with mujoco.Renderer
 * (OpenGL, unavailable here); this is a CUDA ray caster over analytic primitives (DESIGN.md readings
 * Q45-Q48): the floor plane z = 0 seen from above and every OTHER drone of the same env as an oblate spheroid with semi-axes
 * (body_radius, body_radius, body_half_height) in its body frame, front faces only.  Optical axis = body +x, image right =
 * body -y, image up = body +z; fovy_deg is the vertical field of view; pixel (r, c), row 0 at the top, looks along the body
 * direction (1, -(c + 1/2 - width/2) s, -(r + 1/2 - height/2) s), s = 2 tan(fovy/2) / height. */
typedef struct mdg_cam_params {
    uint32_t struct_size;           /* must equal sizeof(mdg_cam_params) (set by mdg_default_cam_params) */
    int32_t height, width;          /* 48, 64; width must be a multiple of 4 */
    float fovy_deg, offset[3];      /* 60; (0.02, 0, 0) m in the body frame */
    float znear, zfar;              /* 0.01, 50 m: hits outside [znear, zfar) are discarded */
    float body_radius, body_half_height;   /* arm + propeller radius of the drone model; 0.0125 m */
} mdg_cam_params;

/* Fill *out with the defaults above (48 x 64, 60 degrees, offset [0.02, 0, 0]); params (host, may be NULL =
 * CF2X) supplies arm length and propeller radius (Table 2).  MDG_EINVAL: NULL out. */
int mdg_default_cam_params(const mdg_params* params, mdg_cam_params* out);

/* Render every drone's camera from the CURRENT state (after the last reset / step on the bound stream; asynchronous on it).
 * cam: host pointer, NULL = defaults for the handle's drone model.  depth_dev: [n_envs*n_drones][height][width] fp32, distance
 * along the optical axis in metres, zfar where nothing is hit; caller-owned device memory, 16-byte aligned.  seg_dev: same
 * shape, u8: 0 background, 1 floor, 2 + k drone k of the env; caller-owned, 4-byte aligned.  Either may be NULL (not written).
 * MDG_EINVAL on a NULL handle, both outputs NULL, misaligned pointers, width % 4 != 0, non-positive sizes, fovy outside
 * (0, 180), znear <= 0 or zfar <= znear, non-positive body axes. */
int mdg_render_depth(mdg_env* env, const mdg_cam_params* cam, float* depth_dev, uint8_t* seg_dev);

/* The colour frame of the same cameras: PAPER.md:177's "(N, 48, 64, 4) uint8" observation, [n_envs*n_drones][height][width][4]
 * u8 = R, G, B, A, caller-owned device memory, 16-byte aligned.  The paper's frame comes from mujoco.Renderer (OpenGL,
 * unavailable here); this one is flat Lambert shading of the hit mdg_render_depth finds (reading Q53): one directional
 * light, unit vector towards it l = (0.36, 0.48, 0.80) in the world frame; shade = 0.3 + 0.7 max(0, n.l), n the outward unit
 * normal at the hit (floor +z; spheroid: normalised gradient of its quadric); albedo 0..255: floor (160, 160, 160), drone k
 * (250 - 22 (k mod 8), 60 + 40 ((k div 8) mod 4), 40 + 26 (k mod 8)); channel = floor(albedo * shade + 1/2) in fp32;
 * background = the unshaded sky (135, 206, 235); A = 255.  Same cam argument, scene, clipping, stream behaviour and errors as
 * mdg_render_depth (MDG_EINVAL also for a NULL or misaligned rgba_dev). */
int mdg_render_rgba(mdg_env* env, const mdg_cam_params* cam, uint8_t* rgba_dev);

/* Bind the CUDA stream (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream) used by later calls.  Work already queued
 * on the previously bound stream (the clear and reset of mdg_create, earlier steps) is ordered before whatever is enqueued on
 * the new one afterwards (an event on the old stream, waited on by the new; skipped when either stream is being captured:
 * inside a capture the ordering is the caller's graph).  MDG_EINVAL: NULL handle.  (The simulator itself has no notion of streams; this serves PAPER.md:292, keeping the loop on the device.) */
int mdg_set_stream(mdg_env* env, void* cuda_stream);

/* Introspection (no counterpart in the paper; bench.py's `gpu_launches` and the tests use them): kernels launched so far
 * through this handle; name of the step kernel specialisation ("step_kernel<G, feature word, blocks/SM[, x2]>", "jit" or
 * "generic" inside it says how it was built; the string lives as long as the handle). */
int64_t mdg_launch_count(const mdg_env* env);
const char* mdg_kernel_name(const mdg_env* env);
/* Launch shape tuning (0 keeps the current value): threads per block (a multiple of 32 in [32, 128]), and a cap on resident blocks
 * per SM (1..32).  Results do not depend on the launch shape.  Drops cached graphs.  MDG_EINVAL: NULL handle, bad block size. */
int mdg_set_launch(mdg_env* env, int block_threads, int max_blocks_per_sm);

/* Measurement aid for the roofline denominator: runs a register-only FFMA kernel (8 independent
 * chains per thread, every SM full) on the current device, times it with CUDA events on `cuda_stream` and writes
 * the achieved FP32 rate in TFLOP/s (2 flop per FFMA) to *tflops (host pointer).  Synchronises the stream. */
int mdg_measure_fp32_peak(void* cuda_stream, double* tflops);

/* Thread-local text of the last failure in this thread (or the note a successful mdg_create left about a kernel fallback);
 * never NULL. */
const char* mdg_last_error(void);
/* Library version; checkpoints of another version are refused by mdg_load. */
int mdg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MDG_H */

// oracle/drone_oracle.hpp — TEST INFRASTRUCTURE: the plain, slow, float64 CPU oracle of the batched
// drone-environment step of arxiv/paper_2606_08039 ("MuJoCo-Drones-Gym").
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
// import, link or execute anything under oracle/.  It shares no code, header, table or constant
// generator with the CUDA path (paper_2606_08039_b200/csrc/, include/mdg.h); the enum VALUES below
// are restated because they are the interface both sides receive from the workload recipes.
//
// The method is a time-stepping iteration, so this file follows the algorithm step by step in the
// paper's order: scalar loops env -> drone, no blocking, no fusion, no reordering.  Each function cites
// the PAPER.md passage it follows; where the paper is silent the reading Qn of SURVEY.md §8(c) /
// DESIGN.md §3 is named.  The scalar type R is a template parameter: R=double is the oracle,
// R=Counted (oracle_capi.cpp) yields the algorithmic flop tally used by bench.py's roofline.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): O1 constants, free fall, hover equilibrium, uniform
// thrust / pure yaw closed forms, torque-free rotation invariants + axisymmetric top + convergence
// order, ground / drag / downwash closed forms, symmetries, PID fixed point + linear z recurrence +
// allocation round trip, wind statistics, obs/reward/termination on hand-built states, Philox KATs;
// tests/test_oracle_next1.py: normalised / one-dimensional / attitude actions, KIN20, CF2P mixing, the
// velocity-tracking and fly-through epilogues, Table 4 factors and initial ranges, constant / sinusoidal wind;
// tests/test_oracle_sensors.py: Table 4 sensor noise and the per-episode observation bias (table standard deviations,
// normality, independence, which columns move, constancy over an episode, keying by global env index);
// tests/test_oracle_dryden.py: altitude-dependent Dryden length scale (printed values, first updates, AR(1) statistics by altitude);
// tests/test_oracle_latency.py: action / sensor latency (thrust-step and free-fall closed forms per substep of delay, shift
// equivalence for the controller action types, uniform per-episode delays);
// tests/test_oracle_formation_path.py: the moving formation centre (hand tables for two polygons, reward / termination about it).
// tests/test_oracle_pid_transient.py: the coupled x / y PID transient against the linearised cascade (a 6-state discrete
// linear system iterated in numpy) at several yaw angles and directions.
// PARITY UNPINNED (the oracle itself is the reference): the large-amplitude (nonlinear) PID transient and the
// multi-config trajectories beyond the invariants above; parity against MuJoCo's own RK4 (MuJoCo is
// not in the container, reading Q11).
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include "philox_ref.hpp"

namespace orc {

// ---- interface enums (values are the interface; Table 1, 179-187 Table 3) -------
enum { AERO_GND = 1, AERO_DRAG = 2, AERO_DW = 4, AERO_WIND = 8 };
enum { INTEG_RK4 = 0, INTEG_EULER = 1 };
enum { PHYS_MJC = 0, PHYS_MJC_GND = 1, PHYS_MJC_DRAG = 2, PHYS_MJC_DW = 3, PHYS_MJC_GND_DRAG_DW = 4, PHYS_DYN = 5 };
enum { ACT_RPM = 0, ACT_PID = 1, ACT_VEL = 2, ACT_RPM_NORM = 3, ACT_ONE_D_RPM = 4, ACT_ATTITUDE = 5 };
enum { OBS_KIN12 = 0, OBS_KIN12_ADJ = 1, OBS_KIN20 = 2, OBS_KIN12_TGT = 3, OBS_KIN12_WP = 4, OBS_KIN12_Z = 5 };
enum { REW_HOVER = 0, REW_NEG_SQ_DIST = 1, REW_MULTI_HOVER = 2, REW_FORMATION = 3, REW_VELOCITY = 4, REW_FLY_THROUGH = 5 };
enum { TERM_NONE = 0, TERM_HOVER = 1, TERM_TILT_DIST = 2, TERM_FORMATION = 3 };
enum { LAYOUT_NONE = 0, LAYOUT_GRID = 1, LAYOUT_CIRCLE = 2 };
enum { TGT_FIXED = 0, TGT_SPAWN_LINSPACE = 1, TGT_BOX = 2, TGT_CIRCLE = 3, TGT_WAYPOINTS = 4 };
enum { MODEL_CF2X = 0, MODEL_CF2P = 1, MODEL_RACE = 2 };

static const double PI = 3.14159265358979323846;

// ---- parameters --------------------------------------------------------------------------------
struct Params {
    // Table 2; units per reading Q1: n in RPM, k_f and k_m per RPM^2.
    double m, g, L, k_f, k_m, J[3], r_p, tw_ratio;
    // aero; values absent from the paper are reading Q5/Q6/Q9.
    double C_gnd, h_clip, c_xy, c_z, dw_C1, dw_C2, dw_C3, dw_dz_clip;
    // wind (readings Q27, Q28)
    double k_wind, wind_sigma, wind_tau;
    int sim_freq, ctrl_freq;
    int aero_mask, integrator;        // -1: take from physics_mode (Table 1)
    // cascaded PID (Table 6; readings Q17-Q21)
    double Kp_pos[3], Ki_pos[3], Kd_pos[3], Kp_att[3], Ki_att[3], Kd_att[3];
    double int_clamp_pos, int_clamp_att;
    int dsl;                          // DSL-PID setpoint rate limits
    double pos_rate_limit, yaw_rate_limit, a_ff[3], tilt_max, tau_xy_max, tau_z_max;
    // observation / reward / termination
    int obs_mode; double adj_radius;
    int reward_mode; double at_target_radius;
    int term_mode; double term_tilt, term_dist, term_center[3], z_max;
    double episode_len_s; int auto_reset;
    // reset distribution and per-episode targets (workload recipe)
    int reset_layout; double reset_center[3], reset_half[3], reset_z_lo, reset_z_hi;
    int grid_cols; double grid_spacing, circle_radius;
    int target_mode; double target_fixed[3], target_lo[3], target_hi[3], mh_z_lo, mh_z_hi,
        form_center[3], form_radius;
    int env_index_base;              // global index of env 0 (sharding across GPUs)
    int drone_model;                 // MODEL_*: CF2P selects the +-configuration mixing (Q37)
    double target_w_lo, target_w_hi; // TGT_BOX: range of the 4th target component (VelocityAviary's yaw rate)
    // Domain randomisation (Table 4): half-widths a of the per-episode multiplicative factors
    // U(1 - a, 1 + a) of [m, J, k_f, k_m, drag c_xy/c_z, C_gnd, downwash C_1, g, per-motor thrust bias (4 draws), arm L,
    // MAX_RPM, -]; all 0 = off (reading Q39).  Initial-state ranges of the same table: RPY_0 and v_0 half-widths.
    double dr_alpha[12];
    double reset_rpy_half[3], reset_vel_half[3];
    // Table 4 "motor lag tau_mot U[5, 50] ms (per ep.)" (reading Q44): first-order rotor-speed lag, time constant drawn per
    // drone and episode from U(motor_lag_lo, motor_lag_hi) seconds; 0, 0 = rotors follow the command at once
    double motor_lag_lo, motor_lag_hi;
    // Wind components (reading Q40): WIND_DRYDEN = the AR(1) gust above, WIND_CONSTANT = steady air
    // velocity wind_const (quadratic drag law), WIND_SINE = the force A [sin wt, cos wt, 0.3 sin 2wt] of episode time t
    int wind_mask; double wind_const[3], wind_sine_amp, wind_sine_omega;
    // WIND_GUST ("random impulses with a smooth sin(pi s) envelope and per-step trigger probability", reading
    // Q42): trigger probability per control step, largest gust speed (m/s), duration of one impulse (s)
    double gust_prob, gust_max, gust_duration;
    // FlyThroughAviary (reading Q41): ordered waypoints, capture radius
    int n_waypoints; double waypoints[24], wp_radius;
    // the waypoint-task family (FlyThroughAviary PAPER.md:321, RaceAviary PAPER.md:329; reading Q43): reward per drone =
    // wp_bonus [capture] - wp_shaping |d_wp| + wp_speed |v| - wp_omega |omega|; the list is run wp_laps times
    double wp_bonus, wp_shaping, wp_speed, wp_omega; int wp_laps;
    // Table 4 "sensors" rows (position / vel / RPY noise N(0, 1 cm / 5 cm/s / 1 deg), gyro noise
    // N(0, 0.05 rad/s), per step) and the "sticky per-episode bias on the observation" of PAPER.md:248 (iii) (reading Q49):
    // standard deviations for [position m, velocity m/s, RPY rad, body rates rad/s]; obs_noise is redrawn every step,
    // obs_bias once per drone and episode; all 0 = off.  Only the emitted observation is perturbed.
    double obs_noise[4], obs_bias[4];
    // DRYDEN with the altitude-dependent length scale ("L_u = h/(0.177 + 8.23e-4 h)^1.2 at altitude h ...
    // alpha = e^(-dt V / L)", reading Q50): V = dryden_airspeed (m/s; 0 = the fixed-tau form above), h = mean altitude of the
    // env's drones at the start of the control step, not below dryden_h_min
    double dryden_airspeed, dryden_h_min;
    // Table 4 latency rows ("action latency U[0, 50] ms (per ep.)", "sensor latency U[0, 20] ms (per ep.)";
    // reading Q51): ranges in seconds, quantised to physics substeps; one delay per drone and episode, uniform over the
    // integers round(lo sim_freq) .. round(hi sim_freq).  Action latency at most 3 control steps, sensor latency at most 1.
    double act_latency_lo, act_latency_hi, obs_latency_lo, obs_latency_hi;
    // FormationAviary's moving centre ("the formation centre tracks a closed polygonal path"; reading Q52): up to 8
    // vertices (x, y, z each), traversed at form_speed m/s from vertex 0 at episode time 0 and closed back to it;
    // form_path_n < 2 or form_speed = 0 = the static centre form_center (Q26)
    int form_path_n; double form_path[24], form_speed;
};
enum { WIND_DRYDEN = 1, WIND_CONSTANT = 2, WIND_GUST = 4, WIND_SINE = 8 };
enum { DR_M = 0, DR_J = 1, DR_KF = 2, DR_KM = 3, DR_DRAG = 4, DR_GND = 5, DR_DW = 6, DR_G = 7, DR_MOTOR = 8 /* 8..11 */, DR_ARM = 12, DR_MAXRPM = 13, DR_LAG = 14 /* tau_mot in seconds, not a factor */, DR_N = 16 };

inline void default_params(int model, Params& P) {
    std::memset(&P, 0, sizeof(P));
    if (model == MODEL_RACE) {        // Table 2, RACE column
        P.m = 0.250; P.L = 0.125; P.tw_ratio = 4.0; P.J[0] = P.J[1] = 4.86e-4; P.J[2] = 8.80e-4;
        P.k_f = 1.28e-8; P.k_m = 5.96e-10; P.r_p = 0.0635;
    } else {                          // Table 2, CF2X column
        P.m = 0.027; P.L = 0.0397; P.tw_ratio = 2.25; P.J[0] = P.J[1] = 1.4e-5; P.J[2] = 2.17e-5;
        P.k_f = 3.16e-10; P.k_m = 7.94e-12; P.r_p = 0.02325;
    }
    P.drone_model = model;
    P.g = 9.81;                                                   // Q2
    P.C_gnd = 11.36859; P.c_xy = 9.1785e-7; P.c_z = 10.311e-7;   // Q5
    P.h_clip = 0.25 * P.r_p * std::sqrt(15.0 * P.C_gnd / 4.0);    // Q6
    P.dw_C1 = 2267.18; P.dw_C2 = 0.16; P.dw_C3 = -0.11;
    P.dw_dz_clip = 0.1;                                           // Q9
    P.k_wind = 0.5 * 1.225 * 1.0 * 0.01;                          // Q28
    P.wind_sigma = 0.5; P.wind_tau = 1.0;
    P.wind_mask = WIND_DRYDEN; P.wind_sine_omega = 2.0 * PI * 0.5;
    P.dryden_airspeed = 0.0; P.dryden_h_min = 0.05;                // Q50
    P.gust_prob = 0.02; P.gust_max = 1.0; P.gust_duration = 0.5;   // Q42
    const double wps[15] = {0, 0, 1, 1, 0, 1, 1, 1, 1.5, 0, 1, 1, 0, 0, 0.5};     // PAPER.md:321 default list
    P.n_waypoints = 5; for (int i = 0; i < 15; ++i) P.waypoints[i] = wps[i];
    P.wp_radius = 0.1;                                            // Q41
    P.wp_bonus = 10.0; P.wp_shaping = 0.1; P.wp_speed = 0.0; P.wp_omega = 0.01; P.wp_laps = 1;
    P.sim_freq = 240; P.ctrl_freq = 48;
    P.aero_mask = -1; P.integrator = -1;
    const double kp[3] = {0.4, 0.4, 1.0}, ki[3] = {0.01, 0.01, 0.01}, kd[3] = {0.9, 0.9, 2.0};     // Table 6
    const double ap[3] = {2e-3, 2e-3, 1e-3}, ai[3] = {0, 0, 1e-4}, ad[3] = {5e-4, 5e-4, 2e-4};
    for (int i = 0; i < 3; ++i) {
        P.Kp_pos[i] = kp[i]; P.Ki_pos[i] = ki[i]; P.Kd_pos[i] = kd[i];
        P.Kp_att[i] = ap[i]; P.Ki_att[i] = ai[i]; P.Kd_att[i] = ad[i];
    }
    P.int_clamp_pos = 2.0; P.int_clamp_att = 0.5; P.dsl = 0;
    P.pos_rate_limit = 2.0; P.yaw_rate_limit = PI; P.tilt_max = 0.5;
    const double s_hover = P.m * P.g / 4.0;                       // Q17
    P.tau_xy_max = 4.0 * (P.L / std::sqrt(2.0)) * s_hover / 3.0;
    if (model == MODEL_CF2P) P.tau_xy_max = 2.0 * P.L * s_hover / 3.0;   // Q37: two rotors per axis, same rule
    P.tau_z_max = 4.0 * (P.k_m / P.k_f) * s_hover / 3.0;
    P.obs_mode = OBS_KIN12; P.adj_radius = 0.5;
    P.reward_mode = REW_HOVER; P.at_target_radius = 0.05;         // Q24
    P.term_mode = TERM_HOVER; P.term_tilt = PI / 2; P.term_dist = 3.0; P.z_max = 3.0;
    P.episode_len_s = 10.0; P.auto_reset = 1;
    P.reset_layout = LAYOUT_NONE; P.reset_center[2] = 1.0;
    P.reset_half[0] = P.reset_half[1] = P.reset_half[2] = 0.1;
    P.grid_cols = 4; P.grid_spacing = 0.3; P.circle_radius = 0.3;
    P.target_mode = TGT_FIXED; P.target_fixed[2] = 1.0;
    P.target_lo[0] = P.target_lo[1] = -1; P.target_lo[2] = 0.2;
    P.target_hi[0] = P.target_hi[1] = 1; P.target_hi[2] = 2.0;
    P.mh_z_lo = 0.7; P.mh_z_hi = 1.2;
    P.form_center[2] = 1.0; P.form_radius = 0.3;                  // PAPER.md:325, Q26
}

// O1 derived constants (reading Q4)
struct Derived {
    double W, hover_rpm, max_rpm, l, kappa, s_max, h, dt_c; int K, ep_steps, aero, integ;
};
inline Derived derive(const Params& P, int physics_mode) {
    Derived d;
    d.W = P.m * P.g;
    d.hover_rpm = std::sqrt(d.W / (4.0 * P.k_f));
    d.max_rpm = std::sqrt(P.tw_ratio * d.W / (4.0 * P.k_f));
    d.l = P.L / std::sqrt(2.0);
    d.kappa = P.k_m / P.k_f;
    d.s_max = P.k_f * d.max_rpm * d.max_rpm;
    d.h = 1.0 / P.sim_freq;
    d.dt_c = 1.0 / P.ctrl_freq;
    d.K = P.sim_freq / P.ctrl_freq;
    d.ep_steps = (int)std::llround(P.episode_len_s * P.ctrl_freq);
    int aero = 0, integ = INTEG_RK4;                              // Table 1
    switch (physics_mode) {
        case PHYS_MJC_GND: aero = AERO_GND; break;
        case PHYS_MJC_DRAG: aero = AERO_DRAG; break;
        case PHYS_MJC_DW: aero = AERO_DW; break;
        case PHYS_MJC_GND_DRAG_DW: aero = AERO_GND | AERO_DRAG | AERO_DW; break;
        case PHYS_DYN: integ = INTEG_EULER; break;
        default: break;
    }
    d.aero = P.aero_mask >= 0 ? P.aero_mask : aero;
    d.integ = P.integrator >= 0 ? P.integrator : integ;
    return d;
}

// Phase marker for the flop tally of oracle_capi.cpp (a no-op for the simulation itself)
#ifndef ORC_PHASE
#define ORC_PHASE(k)
#endif
enum { PH_WIND = 0, PH_DECODE, PH_MOTOR, PH_WRENCH, PH_INTEGRATE, PH_OBS, PH_REWARD, PH_N };

// ---- small linear algebra on scalar type R -----------------------------------------------------
template <class R> inline double to_d(const R& x) { return (double)x; }

// body->world rotation matrix of q=[w,x,y,z]
template <class R> inline void rotmat(const R q[4], R M[3][3]) {
    const R w = q[0], x = q[1], y = q[2], z = q[3];
    M[0][0] = 1.0 - 2.0 * (y * y + z * z); M[0][1] = 2.0 * (x * y - w * z); M[0][2] = 2.0 * (x * z + w * y);
    M[1][0] = 2.0 * (x * y + w * z); M[1][1] = 1.0 - 2.0 * (x * x + z * z); M[1][2] = 2.0 * (y * z - w * x);
    M[2][0] = 2.0 * (x * z - w * y); M[2][1] = 2.0 * (y * z + w * x); M[2][2] = 1.0 - 2.0 * (x * x + y * y);
}
template <class R> inline void mat_vec(const R M[3][3], const R a[3], R out[3]) {
    for (int i = 0; i < 3; ++i) out[i] = M[i][0] * a[0] + M[i][1] * a[1] + M[i][2] * a[2];
}
template <class R> inline void matT_vec(const R M[3][3], const R a[3], R out[3]) {
    for (int i = 0; i < 3; ++i) out[i] = M[0][i] * a[0] + M[1][i] * a[1] + M[2][i] * a[2];
}
template <class R> inline void cross(const R a[3], const R b[3], R out[3]) {
    out[0] = a[1] * b[2] - a[2] * b[1]; out[1] = a[2] * b[0] - a[0] * b[2]; out[2] = a[0] * b[1] - a[1] * b[0];
}
template <class R> inline void quat_mul(const R a[4], const R b[4], R out[4]) {
    out[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    out[1] = a[0] * b[1] + b[0] * a[1] + (a[2] * b[3] - a[3] * b[2]);
    out[2] = a[0] * b[2] + b[0] * a[2] + (a[3] * b[1] - a[1] * b[3]);
    out[3] = a[0] * b[3] + b[0] * a[3] + (a[1] * b[2] - a[2] * b[1]);
}
// Eq.7, readings Q13: Exp(q, phi) = q (x) [cos(|phi|/2), sin(|phi|/2) phi/|phi|];
// phi = omega_body * dt multiplies on the right; series form below 1e-8.
template <class R> inline void quat_exp_step(const R q[4], const R phi[3], R out[4]) {
    const R n2 = phi[0] * phi[0] + phi[1] * phi[1] + phi[2] * phi[2];
    const R n = sqrt(n2);
    R dq[4];
    if (n < 1e-8) {
        dq[0] = 1.0; dq[1] = 0.5 * phi[0]; dq[2] = 0.5 * phi[1]; dq[3] = 0.5 * phi[2];
    } else {
        const R half = 0.5 * n;
        const R s = sin(half) / n;
        dq[0] = cos(half); dq[1] = s * phi[0]; dq[2] = s * phi[1]; dq[3] = s * phi[2];
    }
    quat_mul(q, dq, out);
}
template <class R> inline void quat_normalise(R q[4]) {
    const R n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int i = 0; i < 4; ++i) q[i] = q[i] / n;
}
// ZYX Euler angles (O3.1): roll phi, pitch theta, yaw psi
template <class R> inline void euler_zyx(const R q[4], R eta[3]) {
    const R w = q[0], x = q[1], y = q[2], z = q[3];
    eta[0] = atan2(2.0 * (w * x + y * z), 1.0 - 2.0 * (x * x + y * y));
    R sp = 2.0 * (w * y - z * x);
    if (sp > 1.0) sp = 1.0;
    if (sp < -1.0) sp = -1.0;
    eta[1] = asin(sp);
    eta[2] = atan2(2.0 * (w * z + x * y), 1.0 - 2.0 * (y * y + z * z));
}
template <class R> inline R clampR(const R& x, double lo, double hi) {
    R y = x;
    if (y < lo) y = lo;
    if (y > hi) y = hi;
    return y;
}
template <class R> inline R wrap_pi(const R& x) {     // (-pi, pi]
    const double xd = to_d(x);
    const double k = std::ceil((xd - PI) / (2.0 * PI));
    return x - (2.0 * PI) * k;
}

// ---- per-drone working set ---------------------------------------------------------------------
template <class R> struct Drone {
    R p[3], q[4], v[3], w[3];     // A1 state; w is body-frame (Q22)
    R Ip[3], Ie[3], sp[4];        // PID memory: position / attitude integrals, held setpoint (DSL)
    double tg[4];                 // per-episode target (x, y, z, psi)
    R n_act[4];                   // rotor speeds actually turning (motor lag, Q44); equal to n when the lag is off
    double sc[DR_N];              // domain-randomisation factors of this episode (DR_*; all 1 when off)
    double act[4];                // the action row applied in this control step (KIN20's a_{t-1}); zeros after a reset
    R n[4];                       // rotor speeds in RPM, held over the K substeps (Q21)
    R T, tau_b[3], Om;            // O4: collective thrust, body torque, sum of 2 pi n / 60
    R Fwind[3];                   // O9 wind force, held over the K substeps (Q28)
    R Fw[3], tw[3];               // substep wrench, world frame
    bool hit;                     // sticky floor-hit flag for this control step (Q15)
    double min_abs_pz;            // threshold margin bookkeeping (not part of the method)
};

// PAPER.md:325, reading Q52: centre of the formation at episode time tau, a point moving at constant speed along the closed
// polygon V_0 -> V_1 -> ... -> V_{n-1} -> V_0
inline bool path_on(const Params& P) { return P.target_mode == TGT_CIRCLE && P.form_path_n >= 2 && P.form_speed > 0.0; }
inline void path_centre(const Params& P, double tau, double c[3]) {
    for (int a = 0; a < 3; ++a) c[a] = P.form_center[a];
    if (!path_on(P)) return;
    const int n = P.form_path_n;
    double len[8], perimeter = 0.0;
    for (int k = 0; k < n; ++k) {
        const double* A = &P.form_path[3 * k]; const double* B = &P.form_path[3 * ((k + 1) % n)];
        len[k] = std::sqrt((B[0] - A[0]) * (B[0] - A[0]) + (B[1] - A[1]) * (B[1] - A[1]) + (B[2] - A[2]) * (B[2] - A[2]));
        perimeter += len[k];
    }
    for (int a = 0; a < 3; ++a) c[a] = P.form_path[a];
    if (!(perimeter > 0.0)) return;
    double s = std::fmod(P.form_speed * tau, perimeter);         // arc length travelled on the current lap
    for (int k = 0; k < n; ++k) {
        if (len[k] > 0.0 && (s < len[k] || k == n - 1)) {
            const double* A = &P.form_path[3 * k]; const double* B = &P.form_path[3 * ((k + 1) % n)];
            const double f = s / len[k];
            for (int a = 0; a < 3; ++a) c[a] = A[a] + f * (B[a] - A[a]);
            return;
        }
        s -= len[k];
    }
}

// O4 motor model (Eq.1-3; Q3 yaw pattern m=(1,0,1,0))
template <class R>
inline void motor_wrench(const Params& P, const Derived& D, const R n[4], R& T, R tau[3], R& Om, const double* sc = nullptr) {
    const double kf = sc ? P.k_f * sc[DR_KF] : P.k_f;             // Table 4: k_f, k_m scaled per episode
    const double kappa = sc ? (P.k_m * sc[DR_KM]) / kf : D.kappa;
    const double arm = sc ? sc[DR_ARM] : 1.0;
    R s[4];
    for (int i = 0; i < 4; ++i) s[i] = (sc ? kf * sc[DR_MOTOR + i] : kf) * (n[i] * n[i]);
    T = s[0] + s[1] + s[2] + s[3];
    if (P.drone_model == MODEL_CF2P) {                             // +-configuration (Q37)
        tau[0] = (P.L * arm) * (s[1] - s[3]);
        tau[1] = (P.L * arm) * (s[2] - s[0]);
    } else {
        tau[0] = (D.l * arm) * (s[0] + s[1] - s[2] - s[3]);
        tau[1] = (D.l * arm) * (-s[0] + s[1] + s[2] - s[3]);
    }
    tau[2] = kappa * (-s[0] + s[1] - s[2] + s[3]);
    Om = (2.0 * PI / 60.0) * (n[0] + n[1] + n[2] + n[3]);      // Eq.5's rotor-speed sum
}

// O3.7 closed-form allocation inverse: per-rotor thrusts from (T, tau)
template <class R>
inline void alloc_inverse(const Params& P, const Derived& D, const R& T, const R tau[3], R s[4]) {
    if (P.drone_model == MODEL_CF2P) {                             // inverse of the +-configuration mixing (Q37)
        const R a = tau[0] / P.L, b = tau[1] / P.L, c = tau[2] / D.kappa;
        s[0] = 0.25 * (T - 2.0 * b - c);
        s[1] = 0.25 * (T + 2.0 * a + c);
        s[2] = 0.25 * (T + 2.0 * b - c);
        s[3] = 0.25 * (T - 2.0 * a + c);
        return;
    }
    const R a = tau[0] / D.l, b = tau[1] / D.l, c = tau[2] / D.kappa;
    s[0] = 0.25 * (T + a - b - c);
    s[1] = 0.25 * (T + a + b + c);
    s[2] = 0.25 * (T - a + b - c);
    s[3] = 0.25 * (T - a - b + c);
}

// normalizedActionToRPM (reading Q35): [-1, 1] -> [0, MAX_RPM] through HOVER_RPM at 0, piecewise linear
template <class R>
inline R normalized_to_rpm(const Derived& D, double a_in) {
    const R a = clampR(R(a_in), -1.0, 1.0);
    if (a > 0.0) return D.hover_rpm + (D.max_rpm - D.hover_rpm) * a;
    return (a + 1.0) * D.hover_rpm;
}

// O3.6 attitude PID (D on measurement) and O3.7 allocation inverse with per-rotor clip
template <class R>
inline void attitude_loop_and_mix(const Params& P, const Derived& D, const R& T, const R& phi_ref, const R& th_ref, const R& psi_ref,
                                  const R eta[3], Drone<R>& d) {
    const double dt = D.dt_c;
    R e_eta[3] = {phi_ref - eta[0], th_ref - eta[1], wrap_pi(psi_ref - eta[2])};
    R tau[3];
    for (int i = 0; i < 3; ++i) {
        d.Ie[i] = clampR(d.Ie[i] + e_eta[i] * dt, -P.int_clamp_att, P.int_clamp_att);
        tau[i] = P.Kp_att[i] * e_eta[i] + P.Ki_att[i] * d.Ie[i] - P.Kd_att[i] * d.w[i];
    }
    tau[0] = clampR(tau[0], -P.tau_xy_max, P.tau_xy_max);
    tau[1] = clampR(tau[1], -P.tau_xy_max, P.tau_xy_max);
    tau[2] = clampR(tau[2], -P.tau_z_max, P.tau_z_max);
    R s[4];
    alloc_inverse(P, D, T, tau, s);
    for (int i = 0; i < 4; ++i) d.n[i] = sqrt(clampR(s[i], 0.0, D.s_max) / P.k_f);
}

// O2/O3 action decode -> RPM (Table 3; cascaded PID PAPER.md:347-357, 372-376)
template <class R>
inline void decode_action(const Params& P, const Derived& D, int action_type, const float a_in[4], Drone<R>& d) {
    if (action_type == ACT_RPM) {                                  // Q16: raw RPM, clipped
        for (int i = 0; i < 4; ++i) d.n[i] = clampR(R((double)a_in[i]), 0.0, D.max_rpm);
        return;
    }
    if (action_type == ACT_RPM_NORM || action_type == ACT_ONE_D_RPM) {   // Table 3 / PAPER.md:300, reading Q35
        for (int i = 0; i < 4; ++i) d.n[i] = normalized_to_rpm<R>(D, (double)a_in[action_type == ACT_ONE_D_RPM ? 0 : i]);
        return;
    }
    const double dt = D.dt_c;                                      // Q21: once per control step
    R eta[3];
    euler_zyx(d.q, eta);                                           // O3.1
    const R psi = eta[2];
    if (action_type == ACT_ATTITUDE) {                             // Table 3, reading Q36: [thrust, roll*, pitch*, yaw rate]
        const R nt = normalized_to_rpm<R>(D, (double)a_in[0]);
        const R T = 4.0 * (P.k_f * (nt * nt));
        const R phi_ref = clampR(R((double)a_in[1]), -P.tilt_max, P.tilt_max);
        const R th_ref = clampR(R((double)a_in[2]), -P.tilt_max, P.tilt_max);
        const R psi_ref = psi + (double)a_in[3] * dt;
        attitude_loop_and_mix(P, D, T, phi_ref, th_ref, psi_ref, eta, d);
        return;
    }
    R p_ref[3], v_ref[3], psi_ref;
    if (action_type == ACT_PID) {                                  // O3.2 waypoint [x,y,z,psi]
        const double pc[3] = {(double)a_in[0], (double)a_in[1], (double)a_in[2]};
        const double psic = (double)a_in[3];
        if (P.dsl) {                                               // rate-limited held setpoint
            R dv[3] = {pc[0] - d.sp[0], pc[1] - d.sp[1], pc[2] - d.sp[2]};
            const R dist = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]);
            const double max_step = P.pos_rate_limit * dt;
            if (dist > max_step) {
                const R f = max_step / dist;
                for (int i = 0; i < 3; ++i) d.sp[i] = d.sp[i] + dv[i] * f;
            } else {
                for (int i = 0; i < 3; ++i) d.sp[i] = pc[i];
            }
            R dpsi = wrap_pi(R(psic) - d.sp[3]);
            dpsi = clampR(dpsi, -P.yaw_rate_limit * dt, P.yaw_rate_limit * dt);
            d.sp[3] = wrap_pi(d.sp[3] + dpsi);
        } else {
            for (int i = 0; i < 3; ++i) d.sp[i] = pc[i];
            d.sp[3] = psic;
        }
        for (int i = 0; i < 3; ++i) { p_ref[i] = d.sp[i]; v_ref[i] = 0.0; }
        psi_ref = d.sp[3];
    } else {                                                       // ACT_VEL, Q20: heading frame
        const R c = cos(psi), s = sin(psi);
        const double ax = a_in[0], ay = a_in[1], az = a_in[2], wz = a_in[3];
        for (int i = 0; i < 3; ++i) p_ref[i] = d.p[i];
        v_ref[0] = c * ax - s * ay; v_ref[1] = s * ax + c * ay; v_ref[2] = az;
        psi_ref = psi + wz * dt;
    }
    // O3.3 position loop, Eq.9
    R acc[3];
    for (int i = 0; i < 3; ++i) {
        const R e = p_ref[i] - d.p[i];
        d.Ip[i] = clampR(d.Ip[i] + e * dt, -P.int_clamp_pos, P.int_clamp_pos);
        acc[i] = P.Kp_pos[i] * e + P.Ki_pos[i] * d.Ip[i] + P.Kd_pos[i] * (v_ref[i] - d.v[i]) + P.a_ff[i];
    }
    acc[2] = acc[2] + P.g;
    // O3.4 thrust T = m |a*| (Q18)
    const R T = clampR(P.m * sqrt(acc[0] * acc[0] + acc[1] * acc[1] + acc[2] * acc[2]), 0.0, 4.0 * D.s_max);
    // O3.5 small-angle attitude target (Q17)
    const R cps = cos(psi), sps = sin(psi);
    const R phi_ref = clampR((acc[0] * sps - acc[1] * cps) / P.g, -P.tilt_max, P.tilt_max);
    const R th_ref = clampR((acc[0] * cps + acc[1] * sps) / P.g, -P.tilt_max, P.tilt_max);
    attitude_loop_and_mix(P, D, T, phi_ref, th_ref, psi_ref, eta, d);
}

// O5-O7: world-frame wrench of drone i from the start-of-substep state of all M drones of the env
// (PAPER.md:86-102, 106).
template <class R>
inline void substep_wrench(const Params& P, const Derived& D, Drone<R>* dr, int M, int i) {
    Drone<R>& d = dr[i];
    R Rm[3][3];
    rotmat(d.q, Rm);
    d.Fw[0] = Rm[0][2] * d.T; d.Fw[1] = Rm[1][2] * d.T; d.Fw[2] = Rm[2][2] * d.T;   // R (0,0,T)
    mat_vec(Rm, d.tau_b, d.tw);                                                      // R tau_b
    if (D.aero & AERO_GND) {                       // Eq.4; Q7 body height, Q8 gate R22 > 0
        if (Rm[2][2] > 0.0) {
            R hgt = d.p[2];
            if (hgt < P.h_clip) hgt = P.h_clip;
            const R ratio = P.r_p / (4.0 * hgt);
            d.Fw[2] = d.Fw[2] + (P.C_gnd * d.sc[DR_GND]) * d.T * (ratio * ratio);
        }
    }
    if (D.aero & AERO_DRAG) {                      // Eq.5
        R vb[3], fb[3], fw[3];
        matT_vec(Rm, d.v, vb);
        const double cxy = P.c_xy * d.sc[DR_DRAG], cz = P.c_z * d.sc[DR_DRAG];
        fb[0] = -(cxy * d.Om) * vb[0]; fb[1] = -(cxy * d.Om) * vb[1]; fb[2] = -(cz * d.Om) * vb[2];
        mat_vec(Rm, fb, fw);
        for (int a = 0; a < 3; ++a) d.Fw[a] = d.Fw[a] + fw[a];
    }
    if (D.aero & AERO_DW) {                        // Eq.6 with the regularisation of Q9, reaction per Q10
        for (int k = 0; k < M; ++k) {
            if (k == i) continue;
            const R dz = dr[k].p[2] - d.p[2];
            if (!(dz > 0.0)) continue;
            const R dx = dr[k].p[0] - d.p[0], dy = dr[k].p[1] - d.p[1];
            const R dxy2 = dx * dx + dy * dy;
            if (!(dxy2 < 100.0)) continue;
            R dze = dz, ramp = 1.0;
            if (P.dw_dz_clip > 0.0) {
                if (dze < P.dw_dz_clip) dze = P.dw_dz_clip;
                ramp = dz / P.dw_dz_clip;
                if (ramp > 1.0) ramp = 1.0;
            }
            const R ratio = P.r_p / (4.0 * dze);
            const R alpha = (P.dw_C1 * d.sc[DR_DW]) * (ratio * ratio);
            const R beta = P.dw_C2 * dze + P.dw_C3;
            const R b2 = beta * beta;
            R e;
            if (b2 < 1e-12) e = (to_d(dxy2) == 0.0) ? 1.0 : 0.0;
            else e = exp(-0.5 * dxy2 / b2);
            d.Fw[2] = d.Fw[2] - ramp * alpha * e;
        }
    }
    if (D.aero & AERO_WIND)
        for (int a = 0; a < 3; ++a) d.Fw[a] = d.Fw[a] + d.Fwind[a];
}

// angular acceleration f(q, w) = J^-1 (R(q)^T tau_w - w x J w)  (O8, Q11)
template <class R>
inline void ang_acc(const Params& P, const R q[4], const R w[3], const R tau_w[3], R out[3], double sJ = 1.0) {
    R Rm[3][3], tb[3], Jw[3], c[3];
    rotmat(q, Rm);
    matT_vec(Rm, tau_w, tb);
    for (int a = 0; a < 3; ++a) Jw[a] = (P.J[a] * sJ) * w[a];
    cross(w, Jw, c);
    for (int a = 0; a < 3; ++a) out[a] = (tb[a] - c[a]) / (P.J[a] * sJ);
}

// O8: one physics substep with the wrench frozen in the world frame (Table 1)
template <class R>
inline void integrate(const Params& P, const Derived& D, Drone<R>& d) {
    const double h = D.h;
    const double m = P.m * d.sc[DR_M], g = P.g * d.sc[DR_G], sJ = d.sc[DR_J];
    R a[3] = {d.Fw[0] / m, d.Fw[1] / m, d.Fw[2] / m - g};
    if (D.integ == INTEG_RK4) {
        // translation: classical RK4 on (p, v) with constant acceleration reduces exactly to this
        for (int i = 0; i < 3; ++i) {
            d.p[i] = d.p[i] + h * d.v[i] + (0.5 * h * h) * a[i];
            d.v[i] = d.v[i] + h * a[i];
        }
        // rotation: classical RK4 tableau on (q, w_body), stage orientations by Eq.7 from q0
        R k1[3], k2[3], k3[3], k4[3], q2[4], q3[4], q4[4], w2[3], w3[3], w4[3], ph[3];
        ang_acc(P, d.q, d.w, d.tw, k1, sJ);
        for (int i = 0; i < 3; ++i) { ph[i] = (0.5 * h) * d.w[i]; w2[i] = d.w[i] + (0.5 * h) * k1[i]; }
        quat_exp_step(d.q, ph, q2);
        ang_acc(P, q2, w2, d.tw, k2, sJ);
        for (int i = 0; i < 3; ++i) { ph[i] = (0.5 * h) * w2[i]; w3[i] = d.w[i] + (0.5 * h) * k2[i]; }
        quat_exp_step(d.q, ph, q3);
        ang_acc(P, q3, w3, d.tw, k3, sJ);
        for (int i = 0; i < 3; ++i) { ph[i] = h * w3[i]; w4[i] = d.w[i] + h * k3[i]; }
        quat_exp_step(d.q, ph, q4);
        ang_acc(P, q4, w4, d.tw, k4, sJ);
        for (int i = 0; i < 3; ++i) ph[i] = (h / 6.0) * (d.w[i] + 2.0 * w2[i] + 2.0 * w3[i] + w4[i]);
        R qn[4];
        quat_exp_step(d.q, ph, qn);
        for (int i = 0; i < 3; ++i) d.w[i] = d.w[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
        for (int i = 0; i < 4; ++i) d.q[i] = qn[i];
        quat_normalise(d.q);                                       // Q14
    } else {                                                       // DYN: explicit Euler (Q12)
        for (int i = 0; i < 3; ++i) { d.v[i] = d.v[i] + h * a[i]; d.p[i] = d.p[i] + h * d.v[i]; }
        R k1[3], ph[3], qn[4];
        ang_acc(P, d.q, d.w, d.tw, k1, sJ);                        // R(q0)^T tau_w = tau_b
        for (int i = 0; i < 3; ++i) { d.w[i] = d.w[i] + h * k1[i]; ph[i] = h * d.w[i]; }
        quat_exp_step(d.q, ph, qn);
        for (int i = 0; i < 4; ++i) d.q[i] = qn[i];
        quat_normalise(d.q);
    }
    // floor (Q15)
    const double apz = std::fabs(to_d(d.p[2]));
    if (apz < d.min_abs_pz) d.min_abs_pz = apz;
    if (d.p[2] < 0.0) {
        d.hit = true;
        d.p[2] = 0.0;
        if (d.v[2] < 0.0) d.v[2] = 0.0;
    }
}

// ---- batched simulator ------------------------------------------------------------------------
struct Sim {
    int N, M, physics_mode, action_type;
    Params P; Derived D;
    uint64_t seed; uint32_t gstep;
    std::vector<double> state;    // [D][13] p q v w
    std::vector<double> drs;      // [D][16] domain-randomisation factors of the running episode (DR_*)
    std::vector<double> pid;      // [D][10] Ip Ie sp
    std::vector<double> rotor;    // [D][4] rotor speeds actually turning (RPM), state of the motor lag
    std::vector<double> target;   // [D][4]
    std::vector<double> wind;     // [N][3]
    std::vector<double> gust;     // [N][4] running impulse: velocity vector (m/s) and progress s (>= 1: none)
    std::vector<uint32_t> ep_step;  // [N]
    std::vector<double> obs;      // [N][M*opd]
    std::vector<double> reward;   // [N]
    std::vector<double> reward_d; // [D] per-drone share of the reward (MultiAgentAviary); sums to reward[e]
    std::vector<uint8_t> done;    // [N] bit0 terminated, bit1 truncated
    std::vector<double> margin;   // [N][3] smallest distance to a done / reward / adjacency threshold
    std::vector<float> ahist;     // [D][3][4] the action rows issued 1, 2 and 3 control steps ago (action latency, Q51)

    int opd() const { return P.obs_mode == OBS_KIN20 ? 20 : P.obs_mode == OBS_KIN12_TGT ? 16 : P.obs_mode == OBS_KIN12_WP ? 18 : P.obs_mode == OBS_KIN12_Z ? 13 : 12 + (P.obs_mode == OBS_KIN12_ADJ ? M : 0); }
    int obs_dim() const { return M * opd(); }

    void init(int n_envs, int n_drones, int phys, int act, const Params& p) {
        N = n_envs; M = n_drones; physics_mode = phys; action_type = act; P = p; D = derive(P, phys);
        seed = 0; gstep = 0;
        const size_t Dn = (size_t)N * M;
        state.assign(Dn * 13, 0.0); pid.assign(Dn * 10, 0.0); target.assign(Dn * 4, 0.0); drs.assign(Dn * DR_N, 1.0); rotor.assign(Dn * 4, 0.0);
        wind.assign((size_t)N * 3, 0.0); ep_step.assign(N, 0);
        gust.assign((size_t)N * 4, 0.0); for (int e = 0; e < N; ++e) gust[(size_t)e * 4 + 3] = 1.0;
        obs.assign((size_t)N * obs_dim(), 0.0); reward.assign(N, 0.0); reward_d.assign((size_t)N * M, 0.0); done.assign(N, 0);
        margin.assign((size_t)N * 3, 1e30);
        ahist.assign(Dn * 12, 0.0f);
        for (size_t i = 0; i < Dn; ++i) state[i * 13 + 3] = 1.0;
    }

    // O11/O12: draw the initial state of env e at control-step index t (K2 `_single_reset`)
    void reset_env(int e, uint32_t t) {
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        for (int i = 0; i < M; ++i) {
            const size_t di = (size_t)e * M + i;
            double base[3] = {P.reset_center[0], P.reset_center[1], P.reset_center[2]};
            if (P.reset_layout == LAYOUT_GRID) {
                const int cols = P.grid_cols, rows = (M + cols - 1) / cols;
                base[0] += ((i % cols) - 0.5 * (cols - 1)) * P.grid_spacing;
                base[1] += ((i / cols) - 0.5 * (rows - 1)) * P.grid_spacing;
            } else if (P.reset_layout == LAYOUT_CIRCLE) {
                const double ang = 2.0 * PI * i / M;
                base[0] += P.circle_radius * std::cos(ang);
                base[1] += P.circle_radius * std::sin(ang);
            }
            const PhiloxOut r = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, (uint32_t)i, t, STREAM_RESET_POS, k0, k1);
            double* s = &state[di * 13];
            s[0] = base[0] + (-P.reset_half[0] + 2.0 * P.reset_half[0] * u01(r.x[0]));
            s[1] = base[1] + (-P.reset_half[1] + 2.0 * P.reset_half[1] * u01(r.x[1]));
            if (P.reset_z_hi > P.reset_z_lo) s[2] = P.reset_z_lo + (P.reset_z_hi - P.reset_z_lo) * u01(r.x[2]);
            else s[2] = base[2] + (-P.reset_half[2] + 2.0 * P.reset_half[2] * u01(r.x[2]));
            s[3] = 1.0; s[4] = s[5] = s[6] = 0.0;                   // identity attitude
            for (int a = 7; a < 13; ++a) s[a] = 0.0;                // at rest
            // Table 4 "init" row: RPY_0 and v_0 uniform in +- the given half-widths (0 = the paper's default start)
            if (P.reset_rpy_half[0] != 0.0 || P.reset_rpy_half[1] != 0.0 || P.reset_rpy_half[2] != 0.0) {
                const PhiloxOut rr = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, (uint32_t)i, t, STREAM_INIT_RPY, k0, k1);
                double hr[3];
                for (int a = 0; a < 3; ++a) hr[a] = 0.5 * P.reset_rpy_half[a] * (2.0 * u01(rr.x[a]) - 1.0);   // half angles
                const double cr = std::cos(hr[0]), sr = std::sin(hr[0]), cp = std::cos(hr[1]), sp = std::sin(hr[1]), cy = std::cos(hr[2]), sy = std::sin(hr[2]);
                s[3] = cr * cp * cy + sr * sp * sy; s[4] = sr * cp * cy - cr * sp * sy;     // ZYX: q = q_z(yaw) q_y(pitch) q_x(roll)
                s[5] = cr * sp * cy + sr * cp * sy; s[6] = cr * cp * sy - sr * sp * cy;
            }
            if (P.reset_vel_half[0] != 0.0 || P.reset_vel_half[1] != 0.0 || P.reset_vel_half[2] != 0.0) {
                const PhiloxOut rv = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, (uint32_t)i, t, STREAM_INIT_VEL, k0, k1);
                for (int a = 0; a < 3; ++a) s[7 + a] = P.reset_vel_half[a] * (2.0 * u01(rv.x[a]) - 1.0);
            }
            double* tg = &target[di * 4];
            tg[3] = 0.0;
            if (P.target_mode == TGT_FIXED) {
                tg[0] = P.target_fixed[0]; tg[1] = P.target_fixed[1]; tg[2] = P.target_fixed[2];
            } else if (P.target_mode == TGT_SPAWN_LINSPACE) {
                tg[0] = s[0]; tg[1] = s[1];
                tg[2] = (M > 1) ? P.mh_z_lo + (P.mh_z_hi - P.mh_z_lo) * i / (M - 1) : P.mh_z_lo;
            } else if (P.target_mode == TGT_BOX) {                  // Q32
                const PhiloxOut r2 = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, (uint32_t)i, t, STREAM_RESET_EXTRA, k0, k1);
                for (int a = 0; a < 3; ++a) tg[a] = P.target_lo[a] + (P.target_hi[a] - P.target_lo[a]) * u01(r2.x[a]);
                tg[3] = P.target_w_lo + (P.target_w_hi - P.target_w_lo) * u01(r2.x[3]);
            } else if (P.target_mode == TGT_WAYPOINTS) {            // chase waypoint 0 first; tg[3] = its index
                tg[0] = P.waypoints[0]; tg[1] = P.waypoints[1]; tg[2] = P.waypoints[2];
            } else {                                                // TGT_CIRCLE, Q26
                const double ang = 2.0 * PI * i / M;
                double c[3];
                path_centre(P, 0.0, c);                             // Q52: the path's first vertex when a path is given
                tg[0] = c[0] + P.form_radius * std::cos(ang);
                tg[1] = c[1] + P.form_radius * std::sin(ang);
                tg[2] = c[2];
            }
            // Table 4, Q39: per-episode factors 1 + a (2u - 1); vehicle parameters per drone, g per env
            const bool lag_on = P.motor_lag_hi > 0.0;
            for (int a = 0; a < 4; ++a) rotor[di * 4 + a] = derive(P, 0).hover_rpm;   // Q44: an episode starts with the rotors at hover speed
            bool dr_on = lag_on;
            for (int a = 0; a < 12; ++a) dr_on = dr_on || P.dr_alpha[a] != 0.0;
            if (dr_on) {
                const uint32_t eg = (uint32_t)e + (uint32_t)P.env_index_base;
                const PhiloxOut d0 = philox4x32_10(eg, (uint32_t)i, t, STREAM_DR0, k0, k1);
                const PhiloxOut d1 = philox4x32_10(eg, (uint32_t)i, t, STREAM_DR1, k0, k1);
                const PhiloxOut dg = philox4x32_10(eg, ENV_LEVEL, t, STREAM_DR1, k0, k1);
                const PhiloxOut d2 = philox4x32_10(eg, (uint32_t)i, t, STREAM_DR2, k0, k1);
                const PhiloxOut d3 = philox4x32_10(eg, (uint32_t)i, t, STREAM_DR3, k0, k1);
                double* sc = &drs[di * DR_N];
                for (int a = 0; a < 4; ++a) sc[DR_MOTOR + a] = 1.0 + P.dr_alpha[8] * (2.0 * u01(d2.x[a]) - 1.0);
                sc[DR_ARM] = 1.0 + P.dr_alpha[9] * (2.0 * u01(d3.x[0]) - 1.0);
                sc[DR_MAXRPM] = 1.0 + P.dr_alpha[10] * (2.0 * u01(d3.x[1]) - 1.0);
                sc[DR_LAG] = lag_on ? P.motor_lag_lo + (P.motor_lag_hi - P.motor_lag_lo) * u01(d3.x[2]) : 1.0;
                for (int a = 0; a < 4; ++a) sc[a] = 1.0 + P.dr_alpha[a] * (2.0 * u01(d0.x[a]) - 1.0);
                for (int a = 0; a < 3; ++a) sc[4 + a] = 1.0 + P.dr_alpha[4 + a] * (2.0 * u01(d1.x[a]) - 1.0);
                sc[DR_G] = 1.0 + P.dr_alpha[DR_G] * (2.0 * u01(dg.x[0]) - 1.0);
            }
            double* pm = &pid[di * 10];
            for (int a = 0; a < 6; ++a) pm[a] = 0.0;
            pm[6] = s[0]; pm[7] = s[1]; pm[8] = s[2]; pm[9] = 0.0;  // held setpoint starts at the spawn pose
        }
        wind[(size_t)e * 3 + 0] = wind[(size_t)e * 3 + 1] = wind[(size_t)e * 3 + 2] = 0.0;
        gust[(size_t)e * 4 + 0] = gust[(size_t)e * 4 + 1] = gust[(size_t)e * 4 + 2] = 0.0; gust[(size_t)e * 4 + 3] = 1.0;
        ep_step[e] = 0;
    }

    template <class R> void load(int e, Drone<R>* dr) const {
        for (int i = 0; i < M; ++i) {
            const size_t di = (size_t)e * M + i;
            const double* s = &state[di * 13]; const double* pm = &pid[di * 10];
            Drone<R>& d = dr[i];
            for (int a = 0; a < 3; ++a) { d.p[a] = s[a]; d.v[a] = s[7 + a]; d.w[a] = s[10 + a]; d.Ip[a] = pm[a]; d.Ie[a] = pm[3 + a]; }
            for (int a = 0; a < 4; ++a) { d.q[a] = s[3 + a]; d.sp[a] = pm[6 + a]; d.tg[a] = target[di * 4 + a]; }
            for (int a = 0; a < 3; ++a) d.Fwind[a] = 0.0;
            for (int a = 0; a < 4; ++a) d.act[a] = 0.0;
            for (int a = 0; a < DR_N; ++a) d.sc[a] = drs[di * DR_N + a];
            for (int a = 0; a < 4; ++a) d.n_act[a] = rotor[di * 4 + a];
            d.hit = false; d.min_abs_pz = 1e30;
        }
    }
    template <class R> void store(int e, const Drone<R>* dr) {
        for (int i = 0; i < M; ++i) {
            const size_t di = (size_t)e * M + i;
            double* s = &state[di * 13]; double* pm = &pid[di * 10];
            const Drone<R>& d = dr[i];
            for (int a = 0; a < 3; ++a) { s[a] = to_d(d.p[a]); s[7 + a] = to_d(d.v[a]); s[10 + a] = to_d(d.w[a]); pm[a] = to_d(d.Ip[a]); pm[3 + a] = to_d(d.Ie[a]); }
            for (int a = 0; a < 4; ++a) { s[3 + a] = to_d(d.q[a]); pm[6 + a] = to_d(d.sp[a]); rotor[di * 4 + a] = to_d(d.n_act[a]); }
        }
    }

    // O10: observation of env e from dr (S9: [p, eta, v, w] per drone (+ adjacency row, Q23))
    // Table 4 sensor rows (reading Q49): additive terms nz[12] for [p, eta, v, omega] of drone i of env e in the observation
    // emitted at control-step index t: sigma_g xi (fresh every step) + beta_g b (b drawn at the episode's reset index
    // t0 = t - ep_step).  Twelve normals = three Philox calls, four Box-Muller values each: (x0, x1) -> r cos, r sin; (x2, x3) likewise.
    static void normals4(const PhiloxOut& r, double out[4]) {
        const double r1 = std::sqrt(-2.0 * std::log(1.0 - u01(r.x[0]))), r2 = std::sqrt(-2.0 * std::log(1.0 - u01(r.x[2])));
        out[0] = r1 * std::cos(2.0 * PI * u01(r.x[1])); out[1] = r1 * std::sin(2.0 * PI * u01(r.x[1]));
        out[2] = r2 * std::cos(2.0 * PI * u01(r.x[3])); out[3] = r2 * std::sin(2.0 * PI * u01(r.x[3]));
    }
    void sensor_terms(int e, int i, uint32_t t, double nz[12]) const {
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32), eg = (uint32_t)e + (uint32_t)P.env_index_base;
        const int group[12] = {0, 0, 0, 2, 2, 2, 1, 1, 1, 3, 3, 3};   // [p, eta, v, omega] -> index into (pos, vel, RPY, gyro)
        const uint32_t t0 = t - ep_step[e];                            // index of the reset that opened the running episode
        for (int c = 0; c < 3; ++c) {
            double xi[4], b[4];
            normals4(philox4x32_10(eg, (uint32_t)i, t, STREAM_OBS_NOISE + c, k0, k1), xi);
            normals4(philox4x32_10(eg, (uint32_t)i, t0, STREAM_OBS_BIAS + c, k0, k1), b);
            for (int a = 0; a < 4; ++a) nz[4 * c + a] = P.obs_noise[group[4 * c + a]] * xi[a] + P.obs_bias[group[4 * c + a]] * b[a];
        }
    }
    bool sensors_on() const { for (int a = 0; a < 4; ++a) if (P.obs_noise[a] != 0.0 || P.obs_bias[a] != 0.0) return true; return false; }

    // sensed: the state each drone's kinematic entries are read from (sensor latency, Q51); nullptr = the current state
    template <class R> void write_obs(int e, const Drone<R>* dr_true, double& adj_margin, uint32_t t, const Drone<R>* sensed = nullptr) {
        const int od = opd();
        const bool noisy = sensors_on();
        const Drone<R>* dr = sensed ? sensed : dr_true;             // [p, q, eta, v, omega]; targets are the same in both
        double* o = &obs[(size_t)e * obs_dim()];
        adj_margin = 1e30;
        for (int i = 0; i < M; ++i) {
            R eta[3];
            euler_zyx(dr[i].q, eta);
            double* oi = o + (size_t)i * od;
            if (P.obs_mode == OBS_KIN20) {                         // [p, q, eta, v, omega, a_{t-1}]
                for (int a = 0; a < 3; ++a) { oi[a] = to_d(dr[i].p[a]); oi[7 + a] = to_d(eta[a]); oi[10 + a] = to_d(dr[i].v[a]); oi[13 + a] = to_d(dr[i].w[a]); }
                for (int a = 0; a < 4; ++a) { oi[3 + a] = to_d(dr[i].q[a]); oi[16 + a] = dr[i].act[a]; }
                if (noisy) {                                        // q and the last action stay exact (Q49)
                    double nz[12]; sensor_terms(e, i, t, nz);
                    for (int a = 0; a < 3; ++a) { oi[a] += nz[a]; oi[7 + a] += nz[3 + a]; oi[10 + a] += nz[6 + a]; oi[13 + a] += nz[9 + a]; }
                }
                continue;
            }
            for (int a = 0; a < 3; ++a) { oi[a] = to_d(dr[i].p[a]); oi[3 + a] = to_d(eta[a]); oi[6 + a] = to_d(dr[i].v[a]); oi[9 + a] = to_d(dr[i].w[a]); }
            if (noisy) {                                            // Table 4 sensor rows on the 12 kinematic entries only (Q49)
                double nz[12]; sensor_terms(e, i, t, nz);
                for (int a = 0; a < 12; ++a) oi[a] += nz[a];
            }
            if (P.obs_mode == OBS_KIN12_TGT)                       // [p, eta, v, omega, v*_x, v*_y, v*_z, omega*_z]
                for (int a = 0; a < 4; ++a) oi[12 + a] = dr[i].tg[a];
            if (P.obs_mode == OBS_KIN12_Z) oi[12] = dr[i].tg[2];   // kinematic state plus target altitude (13)
            if (P.obs_mode == OBS_KIN12_WP) {                      // next waypoint and its position in the body frame
                R Rm[3][3], rel[3] = {dr_true[i].tg[0] - dr_true[i].p[0], dr_true[i].tg[1] - dr_true[i].p[1], dr_true[i].tg[2] - dr_true[i].p[2]}, rb[3];
                rotmat(dr_true[i].q, Rm);
                matT_vec(Rm, rel, rb);
                for (int a = 0; a < 3; ++a) { oi[12 + a] = dr_true[i].tg[a]; oi[15 + a] = to_d(rb[a]); }
            }
            if (P.obs_mode == OBS_KIN12_ADJ) {
                for (int k = 0; k < M; ++k) {
                    if (k == i) { oi[12 + k] = 1.0; continue; }
                    const R dx = dr_true[i].p[0] - dr_true[k].p[0], dy = dr_true[i].p[1] - dr_true[k].p[1], dz = dr_true[i].p[2] - dr_true[k].p[2];
                    const R dist = sqrt(dx * dx + dy * dy + dz * dz);
                    oi[12 + k] = (dist < P.adj_radius) ? 1.0 : 0.0;
                    const double mg = std::fabs(to_d(dist) - P.adj_radius);
                    if (mg < adj_margin) adj_margin = mg;
                }
            }
        }
    }

    // one control step of env e (call stack (a)/(b) of SURVEY.md §3)
    template <class R> void step_env(int e, const float* actions, uint32_t t) {
        std::vector<Drone<R>> buf(M);
        Drone<R>* dr = buf.data();
        load(e, dr);
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        // O9 wind gust (PAPER.md:203 recursion, Q27), once per control step, before the substeps
        ORC_PHASE(PH_WIND);
        if (D.aero & AERO_WIND) {
            R w[3] = {0.0, 0.0, 0.0};                              // air velocity seen by the env's drones
            if (P.wind_mask & WIND_DRYDEN) {
                const PhiloxOut r = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, ENV_LEVEL, t, STREAM_WIND, k0, k1);
                const double ua = u01(r.x[0]), ub = u01(r.x[1]), uc = u01(r.x[2]), ud = u01(r.x[3]);
                const R r1 = sqrt(-2.0 * log(R(1.0 - ua))), r2 = sqrt(-2.0 * log(R(1.0 - uc)));   // Box-Muller
                const R xi[3] = {r1 * cos(R(2.0 * PI * ub)), r1 * sin(R(2.0 * PI * ub)), r2 * cos(R(2.0 * PI * ud))};
                double alpha = std::exp(-D.dt_c / P.wind_tau);
                if (P.dryden_airspeed > 0.0) {                     // PAPER.md:202, Q50: L_u(h), alpha = exp(-dt V / L)
                    double hm = 0.0;
                    for (int i = 0; i < M; ++i) hm += to_d(dr[i].p[2]);
                    hm = std::fmax(hm / M, P.dryden_h_min);
                    const double L = hm / std::pow(0.177 + 8.23e-4 * hm, 1.2);
                    alpha = std::exp(-D.dt_c * P.dryden_airspeed / L);
                }
                const double gain = P.wind_sigma * std::sqrt(1.0 - alpha * alpha);
                for (int a = 0; a < 3; ++a) { w[a] = alpha * R(wind[(size_t)e * 3 + a]) + gain * xi[a]; wind[(size_t)e * 3 + a] = to_d(w[a]); }
            }
            if (P.wind_mask & WIND_CONSTANT)                       // steady wind, same quadratic drag law
                for (int a = 0; a < 3; ++a) w[a] = w[a] + P.wind_const[a];
            if (P.wind_mask & WIND_GUST) {                         // PAPER.md:201, Q42
                double* gs = &gust[(size_t)e * 4];
                // an impulse is over once its phase has reached 1 - 1e-4 (Q42): the envelope is 3e-4 there, and a duration that is a
                // whole number of control steps (the default 0.5 s = 24 steps) is not decided by the last bit of the accumulated phase
                constexpr double GUST_END = 1.0 - 1e-4;
                if (gs[3] >= GUST_END) {                           // no impulse running: trigger with probability gust_prob
                    const PhiloxOut r = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, ENV_LEVEL, t, STREAM_GUST, k0, k1);
                    if (u01(r.x[0]) < P.gust_prob) {
                        const double amp = P.gust_max * u01(r.x[1]), z = 2.0 * u01(r.x[2]) - 1.0, ph = 2.0 * PI * u01(r.x[3]);
                        const double rxy = std::sqrt(1.0 - z * z);  // direction uniform on the sphere
                        gs[0] = amp * rxy * std::cos(ph); gs[1] = amp * rxy * std::sin(ph); gs[2] = amp * z; gs[3] = 0.0;
                    }
                }
                if (gs[3] < GUST_END) {                            // smooth envelope sin(pi s), s advancing by dt / duration
                    const R env_s = sin(R(PI * gs[3]));
                    for (int a = 0; a < 3; ++a) w[a] = w[a] + gs[a] * env_s;
                    gs[3] += D.dt_c / P.gust_duration;
                }
            }
            R fs[3] = {0.0, 0.0, 0.0};
            if (P.wind_mask & WIND_SINE) {                         // F(t) = A [sin wt, cos wt, 0.3 sin 2wt]
                const R ph = P.wind_sine_omega * ((double)ep_step[e] * D.dt_c);   // episode time at the start of the step
                fs[0] = P.wind_sine_amp * sin(ph); fs[1] = P.wind_sine_amp * cos(ph); fs[2] = (0.3 * P.wind_sine_amp) * sin(2.0 * ph);
            }
            const bool drag = (P.wind_mask & (WIND_DRYDEN | WIND_CONSTANT | WIND_GUST)) != 0;
            for (int i = 0; i < M; ++i) {                          // PAPER.md:201 drag law, Q28
                R rel[3] = {w[0] - dr[i].v[0], w[1] - dr[i].v[1], w[2] - dr[i].v[2]};
                const R nr = sqrt(rel[0] * rel[0] + rel[1] * rel[1] + rel[2] * rel[2]);
                for (int a = 0; a < 3; ++a) dr[i].Fwind[a] = (drag ? (P.k_wind * nr) * rel[a] : R(0.0)) + fs[a];
            }
        }
        ORC_PHASE(PH_DECODE);
        // Table 4 latency rows (Q51): this episode's delays in physics substeps, drawn at the reset index t0 of the episode
        const bool lat_a = P.act_latency_hi > 0.0, lat_s = P.obs_latency_hi > 0.0;
        std::vector<int> d_act(M, 0), d_obs(M, 0), sw(M, -1);
        std::vector<Drone<R>> later(M), snap(M);                   // rotor commands after the switch; sensed state
        if (lat_a || lat_s) {
            const int a_lo = (int)std::floor(P.act_latency_lo * P.sim_freq + 0.5), a_hi = (int)std::floor(P.act_latency_hi * P.sim_freq + 0.5);
            const int s_lo = (int)std::floor(P.obs_latency_lo * P.sim_freq + 0.5), s_hi = (int)std::floor(P.obs_latency_hi * P.sim_freq + 0.5);
            const uint32_t t0 = (t - 1u) - ep_step[e];
            for (int i = 0; i < M; ++i) {
                const PhiloxOut r = philox4x32_10((uint32_t)e + (uint32_t)P.env_index_base, (uint32_t)i, t0, STREAM_LATENCY, k0, k1);
                d_act[i] = a_lo + (int)(((uint64_t)(r.x[0] >> 8) * (uint64_t)(a_hi - a_lo + 1)) >> 24);   // uniform over a_lo..a_hi
                d_obs[i] = s_lo + (int)(((uint64_t)(r.x[1] >> 8) * (uint64_t)(s_hi - s_lo + 1)) >> 24);
            }
        }
        const bool direct = action_type == ACT_RPM || action_type == ACT_RPM_NORM || action_type == ACT_ONE_D_RPM;
        // O2/O3 decode, O4 motor model
        for (int i = 0; i < M; ++i) {
            const float* a_now = actions + ((size_t)e * M + i) * 4;
            const float* a_first = a_now;                           // the row in effect when the control step starts
            if (lat_a) {
                // The row issued at control step t arrives d substeps later: substep k of step t runs the row of step
                // t + floor((k - d) / K).  With d = (n - 1) K + r, 1 <= r <= K: row t - n for k < r, row t - n + 1 from k = r on.
                // A controller (PID / VEL / ATTITUDE) decodes once per control step, from the row that has arrived by then.
                float* H = &ahist[((size_t)e * M + i) * 12];        // H[0..3] = a_{t-1}, H[4..7] = a_{t-2}, H[8..11] = a_{t-3}
                if (ep_step[e] == 0) for (int r = 0; r < 3; ++r) for (int a = 0; a < 4; ++a) H[4 * r + a] = a_now[a];   // primed with the episode's first row
                const int n = (d_act[i] + D.K - 1) / D.K, r = d_act[i] - (n - 1) * D.K;
                float rows[4][4];
                for (int a = 0; a < 4; ++a) { rows[0][a] = a_now[a]; rows[1][a] = H[a]; rows[2][a] = H[4 + a]; rows[3][a] = H[8 + a]; }
                float first[4], second[4];
                for (int a = 0; a < 4; ++a) { first[a] = rows[n][a]; second[a] = rows[n > 0 ? n - 1 : 0][a]; }
                for (int a = 0; a < 4; ++a) { H[8 + a] = H[4 + a]; H[4 + a] = H[a]; H[a] = a_now[a]; }
                decode_action(P, D, action_type, first, dr[i]);
                if (direct && n >= 1 && r < D.K) {
                    later[i] = dr[i];
                    decode_action(P, D, action_type, second, later[i]);
                    sw[i] = r;
                }
                a_first = nullptr;
            }
            if (a_first) decode_action(P, D, action_type, a_first, dr[i]);
            for (int a = 0; a < 4; ++a) dr[i].act[a] = (double)a_now[a];   // KIN20 reports the row the policy issued
            if (dr[i].sc[DR_MAXRPM] != 1.0)                         // Table 4: the true motor saturation of this episode
                for (int a = 0; a < 4; ++a) {
                    if (dr[i].n[a] > D.max_rpm * dr[i].sc[DR_MAXRPM]) dr[i].n[a] = D.max_rpm * dr[i].sc[DR_MAXRPM];
                    if (sw[i] >= 0 && later[i].n[a] > D.max_rpm * dr[i].sc[DR_MAXRPM]) later[i].n[a] = D.max_rpm * dr[i].sc[DR_MAXRPM];
                }
            ORC_PHASE(PH_MOTOR);
            motor_wrench(P, D, dr[i].n, dr[i].T, dr[i].tau_b, dr[i].Om, dr[i].sc);
            ORC_PHASE(PH_DECODE);
        }
        if (lat_s) for (int i = 0; i < M; ++i) if (d_obs[i] >= D.K) snap[i] = dr[i];   // a full step old: the state the step starts from
        // K substeps: all wrenches from the same start-of-substep state, then integrate
        const bool lag = P.motor_lag_hi > 0.0;
        for (int k = 0; k < D.K; ++k) {
            ORC_PHASE(PH_MOTOR);
            for (int i = 0; i < M; ++i)
                if (sw[i] == k) {                                  // Q51: the next row arrives at this substep
                    for (int a = 0; a < 4; ++a) dr[i].n[a] = later[i].n[a];
                    motor_wrench(P, D, dr[i].n, dr[i].T, dr[i].tau_b, dr[i].Om, dr[i].sc);
                }
            if (lag)                                               // Q44: n <- n + (1 - e^(-h/tau)) (n_cmd - n), then Eq.1-3 with n
                for (int i = 0; i < M; ++i) {
                    const double gam = 1.0 - std::exp(-D.h / dr[i].sc[DR_LAG]);
                    for (int a = 0; a < 4; ++a) dr[i].n_act[a] = dr[i].n_act[a] + gam * (dr[i].n[a] - dr[i].n_act[a]);
                    motor_wrench(P, D, dr[i].n_act, dr[i].T, dr[i].tau_b, dr[i].Om, dr[i].sc);
                }
            ORC_PHASE(PH_WRENCH);
            for (int i = 0; i < M; ++i) substep_wrench(P, D, dr, M, i);
            ORC_PHASE(PH_INTEGRATE);
            for (int i = 0; i < M; ++i) integrate(P, D, dr[i]);
            if (lat_s) for (int i = 0; i < M; ++i) if (k + 1 == D.K - d_obs[i]) snap[i] = dr[i];   // what the sensors report d_obs substeps later
        }
        store(e, dr);
        ORC_PHASE(PH_REWARD);
        // O10 reward / termination from the end-of-step state
        const bool use_floor = P.term_mode == TERM_HOVER || P.term_mode == TERM_FORMATION;
        const bool use_tilt = P.term_mode != TERM_NONE;
        const bool use_zmax = use_floor;
        const bool use_dist = P.term_mode == TERM_TILT_DIST || P.term_mode == TERM_FORMATION;
        double centre[3] = {P.term_center[0], P.term_center[1], P.term_center[2]};
        if (path_on(P)) {                                          // PAPER.md:325, Q52: slots ride on the moving centre; evaluated at the end-of-step time
            path_centre(P, (double)(ep_step[e] + 1u) * D.dt_c, centre);
            for (int i = 0; i < M; ++i) {
                const double ang = 2.0 * PI * i / M;
                double* tgs = &target[((size_t)e * M + i) * 4];
                tgs[0] = dr[i].tg[0] = centre[0] + P.form_radius * std::cos(ang);
                tgs[1] = dr[i].tg[1] = centre[1] + P.form_radius * std::sin(ang);
                tgs[2] = dr[i].tg[2] = centre[2];
            }
        }
        double m_done = 1e30, m_rew = 1e30;
        bool terminated = false;
        R rew = 0.0;
        double* rd = &reward_d[(size_t)e * M];                   // bookkeeping beside the env reward, not part of its arithmetic
        for (int i = 0; i < M; ++i) rd[i] = 0.0;
        for (int i = 0; i < M; ++i) {
            const Drone<R>& d = dr[i];
            R eta[3];
            euler_zyx(d.q, eta);
            const R aphi = fabs(eta[0]), ath = fabs(eta[1]);
            bool crash = false;
            if (use_floor) { if (d.hit) { terminated = true; crash = true; } if (d.min_abs_pz < m_done) m_done = d.min_abs_pz; }
            if (use_tilt) {                                         // PAPER.md:309 / config 3
                if (aphi > P.term_tilt || ath > P.term_tilt) { terminated = true; crash = true; }
                m_done = std::fmin(m_done, std::fmin(std::fabs(to_d(aphi) - P.term_tilt), std::fabs(to_d(ath) - P.term_tilt)));
            }
            if (use_zmax) {
                if (d.p[2] > P.z_max) terminated = true;
                m_done = std::fmin(m_done, std::fabs(to_d(d.p[2]) - P.z_max));
            }
            if (use_dist) {
                const R dx = d.p[0] - centre[0], dy = d.p[1] - centre[1], dz = d.p[2] - centre[2];   // the moving centre when a path is on
                const R dist = sqrt(dx * dx + dy * dy + dz * dz);
                if (dist > P.term_dist) terminated = true;
                m_done = std::fmin(m_done, std::fabs(to_d(dist) - P.term_dist));
            }
            const R ex = d.p[0] - d.tg[0], ey = d.p[1] - d.tg[1], ez = d.p[2] - d.tg[2];
            if (P.reward_mode == REW_HOVER || P.reward_mode == REW_MULTI_HOVER) {      // Eq.8, 317
                const R dist = sqrt(ex * ex + ey * ey + ez * ez);
                const R speed = sqrt(d.v[0] * d.v[0] + d.v[1] * d.v[1] + d.v[2] * d.v[2]);
                R r = -fabs(ez) - 0.1 * sqrt(ex * ex + ey * ey) - 0.05 * speed - 0.05 * (aphi + ath);
                if (dist < P.at_target_radius) r = r + 0.5;
                if (crash) r = r - 100.0;
                m_rew = std::fmin(m_rew, std::fabs(to_d(dist) - P.at_target_radius));
                rew = rew + r; rd[i] += to_d(r);
            } else if (P.reward_mode == REW_NEG_SQ_DIST) {          // config 3
                rew = rew - (ex * ex + ey * ey + ez * ez); rd[i] -= to_d(ex * ex + ey * ey + ez * ez);
            } else if (P.reward_mode == REW_VELOCITY) {             // VelocityAviary, target = (v*, omega_z*), Q38
                const R ux = d.v[0] - d.tg[0], uy = d.v[1] - d.tg[1], uz = d.v[2] - d.tg[2];
                const R verr = sqrt(ux * ux + uy * uy + uz * uz);
                R r = -verr - 0.1 * fabs(d.w[2] - d.tg[3]) - 0.05 * (aphi + ath);
                if (verr < P.at_target_radius) r = r + 0.5;
                m_rew = std::fmin(m_rew, std::fabs(to_d(verr) - P.at_target_radius));
                rew = rew + r; rd[i] += to_d(r);
            } else if (P.reward_mode == REW_FLY_THROUGH) {          // PAPER.md:321, Q41
                const R dist = sqrt(ex * ex + ey * ey + ez * ez);   // to the waypoint being chased
                const R wn = sqrt(d.w[0] * d.w[0] + d.w[1] * d.w[1] + d.w[2] * d.w[2]);
                const R speed = sqrt(d.v[0] * d.v[0] + d.v[1] * d.v[1] + d.v[2] * d.v[2]);
                R r = P.wp_speed * speed - P.wp_shaping * dist - P.wp_omega * wn;
                const double mg = std::fabs(to_d(dist) - P.wp_radius);
                m_rew = std::fmin(m_rew, mg); m_done = std::fmin(m_done, mg);
                if (dist < P.wp_radius) {                           // capture: +10, move on; the last one ends the episode
                    r = r + P.wp_bonus;
                    const int k = (int)dr[i].tg[3] + 1;             // running index over all laps
                    if (k >= P.n_waypoints * P.wp_laps) terminated = true;
                    else {
                        const int kw = k % P.n_waypoints;
                        double* tgs = &target[((size_t)e * M + i) * 4];
                        tgs[0] = dr[i].tg[0] = P.waypoints[3 * kw]; tgs[1] = dr[i].tg[1] = P.waypoints[3 * kw + 1];
                        tgs[2] = dr[i].tg[2] = P.waypoints[3 * kw + 2]; tgs[3] = dr[i].tg[3] = (double)k;
                    }
                }
                rew = rew + r; rd[i] += to_d(r);
            } else {                                                // REW_FORMATION (Q26)
                rew = rew - sqrt(ex * ex + ey * ey + ez * ez); rd[i] -= to_d(sqrt(ex * ex + ey * ey + ez * ez));
                for (int k = i + 1; k < M; ++k) {
                    const R ax = d.p[0] - dr[k].p[0], ay = d.p[1] - dr[k].p[1], az = d.p[2] - dr[k].p[2];
                    const double bx = d.tg[0] - dr[k].tg[0], by = d.tg[1] - dr[k].tg[1], bz = d.tg[2] - dr[k].tg[2];
                    const R dact = sqrt(ax * ax + ay * ay + az * az);
                    const double ddes = std::sqrt(bx * bx + by * by + bz * bz);
                    rew = rew - 0.5 * fabs(dact - ddes);
                    rd[i] -= 0.25 * std::fabs(to_d(dact) - ddes); rd[k] -= 0.25 * std::fabs(to_d(dact) - ddes);   // half of the pair term each
                }
            }
        }
        ep_step[e] += 1;
        const bool truncated = D.ep_steps > 0 && (int)ep_step[e] >= D.ep_steps;
        reward[e] = to_d(rew);
        done[e] = (uint8_t)((terminated ? 1 : 0) | (truncated ? 2 : 0));
        // O11 auto-reset (Q29): reward/done describe the finished transition, obs opens the new episode
        bool fresh = false;
        if (done[e] && P.auto_reset) {
            reset_env(e, t);
            load(e, dr);
            fresh = true;                                          // the new episode's first row is its initial state
        }
        double m_adj;
        ORC_PHASE(PH_OBS);
        if (lat_s && !fresh) {
            for (int i = 0; i < M; ++i) { for (int a = 0; a < 4; ++a) { snap[i].tg[a] = dr[i].tg[a]; snap[i].act[a] = dr[i].act[a]; } }
            write_obs(e, dr, m_adj, t, snap.data());
        } else
        write_obs(e, dr, m_adj, t);
        margin[(size_t)e * 3 + 0] = m_done; margin[(size_t)e * 3 + 1] = m_rew; margin[(size_t)e * 3 + 2] = m_adj;
    }

    void reset_all(uint64_t s) {
        seed = s; gstep = 0;
        std::vector<Drone<double>> buf(M);
        for (int e = 0; e < N; ++e) {
            reset_env(e, 0);
            load(e, buf.data());
            double m_adj;
            write_obs(e, buf.data(), m_adj, 0);
            reward[e] = 0.0; done[e] = 0;
            margin[(size_t)e * 3 + 0] = margin[(size_t)e * 3 + 1] = 1e30; margin[(size_t)e * 3 + 2] = m_adj;
        }
    }
    template <class R> void step_range(int e0, int e1, const float* actions, uint32_t t) {
        for (int e = e0; e < e1; ++e) step_env<R>(e, actions, t);
    }
};

}  // namespace orc

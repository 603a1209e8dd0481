// mdg_step.cuh — the fused control-step kernel: one thread per drone, the G = pow2 >= M drones of an
// env sit in adjacent lanes of one warp, the 13 state words stay in registers over all K substeps,
// and every intra-env exchange (downwash pairs, adjacency, reward / done reduction) is a warp shuffle.
// No shared memory, no HBM traffic between substeps.  PAPER.md citations: see include/mdg.h.
#pragma once
#include "mdg_dev.cuh"

namespace mdg {

#define MDG_FULL 0xffffffffu

template <int FEAT> struct Feat {
    __device__ __forceinline__ static int word(const DevParams& P) { return FEAT >= 0 ? FEAT : P.feat; }
    __device__ __forceinline__ static bool has(const DevParams& P, int bit) { return (word(P) & bit) != 0; }
    __device__ __forceinline__ static int act(const DevParams& P) { return (word(P) >> F_ACT_SHIFT) & 7; }
    __device__ __forceinline__ static int rew(const DevParams& P) { return (word(P) >> F_REW_SHIFT) & 7; }
    __device__ __forceinline__ static int obs(const DevParams& P) { return (word(P) >> F_OBS_SHIFT) & 7; }   // MDG_OBS_*
    __device__ __forceinline__ static int term(const DevParams& P) { return (word(P) >> F_TERM_SHIFT) & 3; }
};

struct DroneRegs {
    V3 p; Q4 q; V3 v; V3 w;       // state, w in the body frame
    V3 Ip, Ie; float4 sp;         // controller memory
};

// Initial state of drone j of env e at control-step index t (the paper's `_single_reset`)
__device__ __forceinline__ void reset_drone(const DevParams& P, uint32_t e, uint32_t j, uint32_t t,
                                            DroneRegs& d, float4& tg) {
    float bx = P.reset_center[0], by = P.reset_center[1], bz = P.reset_center[2];
    if (P.reset_layout == 1) {            // GRID
        const int col = (int)j % P.grid_cols, row = (int)j / P.grid_cols;
        bx += ((float)col - 0.5f * (float)(P.grid_cols - 1)) * P.grid_spacing;
        by += ((float)row - 0.5f * (float)(P.grid_rows - 1)) * P.grid_spacing;
    } else if (P.reset_layout == 2) {     // CIRCLE
        float s, c;
        sincospif(2.0f * (float)j / (float)P.M, &s, &c);
        bx = fmaf(P.circle_radius, c, bx); by = fmaf(P.circle_radius, s, by);
    }
    const uint4 r = philox4x32_10(e + P.env_base, j, t, STREAM_RESET_POS, P.seed_lo, P.seed_hi);
    d.p.x = bx + fmaf(2.0f * P.reset_half[0], u01(r.x), -P.reset_half[0]);
    d.p.y = by + fmaf(2.0f * P.reset_half[1], u01(r.y), -P.reset_half[1]);
    if (P.reset_z_hi > P.reset_z_lo) d.p.z = fmaf(P.reset_z_hi - P.reset_z_lo, u01(r.z), P.reset_z_lo);
    else d.p.z = bz + fmaf(2.0f * P.reset_half[2], u01(r.z), -P.reset_half[2]);
    d.q.w = 1.0f; d.q.x = d.q.y = d.q.z = 0.0f;
    d.v = v3(0, 0, 0); d.w = v3(0, 0, 0);
    if (P.reset_rpy_half[0] != 0.0f || P.reset_rpy_half[1] != 0.0f || P.reset_rpy_half[2] != 0.0f) {   // Table 4 "init" row
        const uint4 rr = philox4x32_10(e + P.env_base, j, t, STREAM_INIT_RPY, P.seed_lo, P.seed_hi);
        float sr, cr, sp, cp, sy, cy;
        sincosf(0.5f * P.reset_rpy_half[0] * fmaf(2.0f, u01(rr.x), -1.0f), &sr, &cr);
        sincosf(0.5f * P.reset_rpy_half[1] * fmaf(2.0f, u01(rr.y), -1.0f), &sp, &cp);
        sincosf(0.5f * P.reset_rpy_half[2] * fmaf(2.0f, u01(rr.z), -1.0f), &sy, &cy);
        d.q.w = cr * cp * cy + sr * sp * sy; d.q.x = sr * cp * cy - cr * sp * sy;       // ZYX: q = q_z(yaw) q_y(pitch) q_x(roll)
        d.q.y = cr * sp * cy + sr * cp * sy; d.q.z = cr * cp * sy - sr * sp * cy;
    }
    if (P.reset_vel_half[0] != 0.0f || P.reset_vel_half[1] != 0.0f || P.reset_vel_half[2] != 0.0f) {
        const uint4 rv = philox4x32_10(e + P.env_base, j, t, STREAM_INIT_VEL, P.seed_lo, P.seed_hi);
        d.v = v3(P.reset_vel_half[0] * fmaf(2.0f, u01(rv.x), -1.0f), P.reset_vel_half[1] * fmaf(2.0f, u01(rv.y), -1.0f),
                 P.reset_vel_half[2] * fmaf(2.0f, u01(rv.z), -1.0f));
    } d.Ip = v3(0, 0, 0); d.Ie = v3(0, 0, 0);
    d.sp = make_float4(d.p.x, d.p.y, d.p.z, 0.0f);
    tg.w = 0.0f;
    if (P.target_mode == 0) {             // FIXED
        tg.x = P.target_fixed[0]; tg.y = P.target_fixed[1]; tg.z = P.target_fixed[2];
    } else if (P.target_mode == 1) {      // SPAWN_LINSPACE
        tg.x = d.p.x; tg.y = d.p.y;
        tg.z = P.M > 1 ? fmaf(P.mh_z_hi - P.mh_z_lo, (float)j / (float)(P.M - 1), P.mh_z_lo) : P.mh_z_lo;
    } else if (P.target_mode == 2) {      // BOX
        const uint4 r2 = philox4x32_10(e + P.env_base, j, t, STREAM_RESET_EXTRA, P.seed_lo, P.seed_hi);
        tg.x = fmaf(P.target_hi[0] - P.target_lo[0], u01(r2.x), P.target_lo[0]);
        tg.y = fmaf(P.target_hi[1] - P.target_lo[1], u01(r2.y), P.target_lo[1]);
        tg.z = fmaf(P.target_hi[2] - P.target_lo[2], u01(r2.z), P.target_lo[2]);
        tg.w = fmaf(P.target_w_hi - P.target_w_lo, u01(r2.w), P.target_w_lo);
    } else if (P.target_mode == 4) {      // WAYPOINTS: chase waypoint 0 first
        tg.x = P.waypoints[0]; tg.y = P.waypoints[1]; tg.z = P.waypoints[2];
    } else {                              // CIRCLE slots
        float s, c;
        sincospif(2.0f * (float)j / (float)P.M, &s, &c);
        const bool path = (P.feat & F_PATH) != 0;             // DESIGN.md Q52: an episode starts at the path's first vertex
        tg.x = fmaf(P.form_radius, c, path ? P.path[0] : P.form_center[0]); tg.y = fmaf(P.form_radius, s, path ? P.path[1] : P.form_center[1]);
        tg.z = path ? P.path[2] : P.form_center[2];
    }
}

// PAPER.md:325 (Q52): centre of the formation after ep control steps of the episode, moving at constant speed along the
// closed polygon path[0] -> path[1] -> ... -> path[0]
__device__ __forceinline__ V3 path_centre(const DevParams& P, uint32_t ep) {
    float s = fmodf(P.path_rate * (float)ep, P.path_perimeter);
    V3 c = v3(P.path[0], P.path[1], P.path[2]);
    bool found = false;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        if (k < P.path_n && !found) {
            const float len = P.path_len[k];
            if (len > 0.0f && (s < len || k == P.path_n - 1)) {
                const int kn = (k + 1 == P.path_n) ? 0 : k + 1;
                const float f = s / len;
                c = v3(fmaf(f, P.path[3 * kn] - P.path[3 * k], P.path[3 * k]), fmaf(f, P.path[3 * kn + 1] - P.path[3 * k + 1], P.path[3 * k + 1]),
                       fmaf(f, P.path[3 * kn + 2] - P.path[3 * k + 2], P.path[3 * k + 2]));
                found = true;
            }
            s -= len;
        }
    }
    return c;
}

// normalizedActionToRPM: [-1, 1] -> [0, MAX_RPM] through HOVER_RPM at 0, piecewise linear, clipped
__device__ __forceinline__ float norm_rpm(const DevParams& P, float a) {
    a = clampf(a, -1.0f, 1.0f);
    return a > 0.0f ? fmaf(P.rpm_span, a, P.hover_rpm) : fmaf(a, P.hover_rpm, P.hover_rpm);
}

// Domain-randomisation factors of a new episode (Table 4; vehicle factors per drone, g per env)
__device__ __forceinline__ void draw_dr(const DevParams& P, uint32_t e, uint32_t j, uint32_t t, float4& r0, float4& r1, float4& r2, float4& r3) {
    const uint4 a = philox4x32_10(e + P.env_base, j, t, STREAM_DR0, P.seed_lo, P.seed_hi);
    const uint4 b = philox4x32_10(e + P.env_base, j, t, STREAM_DR1, P.seed_lo, P.seed_hi);
    const uint4 c = philox4x32_10(e + P.env_base, j, t, STREAM_DR2, P.seed_lo, P.seed_hi);
    const uint4 d = philox4x32_10(e + P.env_base, j, t, STREAM_DR3, P.seed_lo, P.seed_hi);
    const uint4 g = philox4x32_10(e + P.env_base, 0xFFFFFFFFu, t, STREAM_DR1, P.seed_lo, P.seed_hi);
    auto f = [](float alpha, uint32_t x) { return fmaf(alpha, fmaf(2.0f, u01(x), -1.0f), 1.0f); };
    r0 = make_float4(f(P.dr_alpha[0], a.x), f(P.dr_alpha[1], a.y), f(P.dr_alpha[2], a.z), f(P.dr_alpha[3], a.w));
    r1 = make_float4(f(P.dr_alpha[4], b.x), f(P.dr_alpha[5], b.y), f(P.dr_alpha[6], b.z), f(P.dr_alpha[7], g.x));
    r2 = make_float4(f(P.dr_alpha[8], c.x), f(P.dr_alpha[8], c.y), f(P.dr_alpha[8], c.z), f(P.dr_alpha[8], c.w));
    r3 = make_float4(f(P.dr_alpha[9], d.x), f(P.dr_alpha[10], d.y),
                     P.motor_lag_hi > 0.0f ? fmaf(P.motor_lag_hi - P.motor_lag_lo, u01(d.z), P.motor_lag_lo) : 1.0f, 1.0f);
}

// Action decode -> per-rotor RPM (Table 3; cascaded PID PAPER.md:347-357, DSL PAPER.md:372-376), in two parts.
// decode_front (per env slot, scalar): rotor-command actions are finished here (returns false); for the controller actions it
// leaves what the loops need in a DecodeMid - roll, pitch and the heading direction of the current attitude, the position error
// and commanded velocity (PID / VEL) or thrust and tilt targets (ATTITUDE), the yaw error - and moves the held setpoint (DSL).
// control_loops (lane-generic, mdg_dev.cuh: one env per lane or two as packed pairs): Eq.9, T = m |a*|, the small-angle tilt
// target, the attitude PID with its clamps, the closed-form allocation inverse and the per-rotor clip.
struct DecodeMid {
    float roll, pitch, cpsi, spsi;        // current attitude: eta_x, eta_y, heading (cos psi, sin psi)
    V3 e_p, v_cmd;                        // position error; commanded velocity in the heading frame (VEL) or zero (PID)
    float e_psi, T, phi_ref, th_ref;      // yaw error; ATTITUDE only: thrust and tilt targets
};
template <int FEAT>
__device__ __forceinline__ bool decode_front(const DevParams& P, float4 a, DroneRegs& d, float n[4], DecodeMid& m) {
    const int act = Feat<FEAT>::act(P);
    if (act == 0) {                       // RPM, clipped
        n[0] = clampf(a.x, 0.0f, P.max_rpm); n[1] = clampf(a.y, 0.0f, P.max_rpm);
        n[2] = clampf(a.z, 0.0f, P.max_rpm); n[3] = clampf(a.w, 0.0f, P.max_rpm);
        return false;
    }
    if (act == 3 || act == 4) {           // RPM_NORM / ONE_D_RPM through normalizedActionToRPM (Q35)
        n[0] = norm_rpm(P, a.x);
        n[1] = act == 4 ? n[0] : norm_rpm(P, a.y); n[2] = act == 4 ? n[0] : norm_rpm(P, a.z); n[3] = act == 4 ? n[0] : norm_rpm(P, a.w);
        return false;
    }
    // roll, pitch and the heading direction (cos psi, sin psi) = normalised (1 - 2(y^2+z^2), 2(wz+xy))
    m.roll = roll_of(d.q);
    m.pitch = pitch_of(d.q);
    const float hc = fmaf(-2.0f, fmaf(d.q.y, d.q.y, __fmul_rn(d.q.z, d.q.z)), 1.0f), hs = __fmul_rn(2.0f, fmaf(d.q.w, d.q.z, __fmul_rn(d.q.x, d.q.y)));
    const float hn2 = fmaf(hc, hc, __fmul_rn(hs, hs));
    const float hr = hn2 > 1e-30f ? rsqrt_fast(hn2) : 0.0f;
    m.cpsi = hn2 > 1e-30f ? __fmul_rn(hc, hr) : 1.0f; m.spsi = __fmul_rn(hs, hr);
    m.e_p = v3(0, 0, 0); m.v_cmd = v3(0, 0, 0); m.T = 0.0f; m.phi_ref = 0.0f; m.th_ref = 0.0f;
    if (act == 5) {                       // ATTITUDE [thrust, roll*, pitch*, yaw rate] (Q36): attitude loop + mixer only
        const float nt = norm_rpm(P, a.x);
        m.T = __fmul_rn(4.0f, __fmul_rn(P.k_f, __fmul_rn(nt, nt)));
        m.phi_ref = clampf(a.y, -P.tilt_max, P.tilt_max);
        m.th_ref = clampf(a.z, -P.tilt_max, P.tilt_max);
        m.e_psi = wrap_pi(__fmul_rn(a.w, P.dt_c));
    } else if (act == 1) {                // PID waypoint [x, y, z, psi]
        if (Feat<FEAT>::has(P, F_DSL)) {
            const V3 dv = v3(__fsub_rn(a.x, d.sp.x), __fsub_rn(a.y, d.sp.y), __fsub_rn(a.z, d.sp.z));
            const float dist = sqrtf(fmaf(dv.x, dv.x, fmaf(dv.y, dv.y, __fmul_rn(dv.z, dv.z))));
            if (dist > P.pos_step_max) {
                const float f = __fdiv_rn(P.pos_step_max, dist);
                d.sp.x = fmaf(dv.x, f, d.sp.x); d.sp.y = fmaf(dv.y, f, d.sp.y); d.sp.z = fmaf(dv.z, f, d.sp.z);
            } else { d.sp.x = a.x; d.sp.y = a.y; d.sp.z = a.z; }
            const float dpsi = clampf(wrap_pi(__fsub_rn(a.w, d.sp.w)), -P.yaw_step_max, P.yaw_step_max);
            d.sp.w = wrap_pi(__fadd_rn(d.sp.w, dpsi));
        } else d.sp = a;
        m.e_p = v3(__fsub_rn(d.sp.x, d.p.x), __fsub_rn(d.sp.y, d.p.y), __fsub_rn(d.sp.z, d.p.z));
        m.e_psi = wrap_pi(__fsub_rn(d.sp.w, atan2_fast(hs, hc)));
    } else {                              // VEL [vx, vy, vz, wz] in the heading frame
        m.v_cmd = v3(a.x, a.y, a.z);
        m.e_psi = wrap_pi(__fmul_rn(a.w, P.dt_c));                 // psi* = psi + wz dt
    }
    return true;
}
template <class T> struct DecodeMidT {   // DecodeMid of one env slot (float) or of the lane's two (F2)
    T roll, pitch, cpsi, spsi, ncpsi, nspsi; V3T<T> e_p, v_cmd; T e_psi, thrust, phi_ref, th_ref;
};
template <int FEAT, class T>
__device__ __forceinline__ void control_loops(const DevParams& P, const DecodeMidT<T>& m, V3T<T> v, V3T<T> w, V3T<T>& Ip, V3T<T>& Ie, T (&n)[4]) {
    const int act = Feat<FEAT>::act(P);
    T thrust = m.thrust, phi_ref = m.phi_ref, th_ref = m.th_ref;
    if (act != 5) {
        // commanded velocity from the heading frame to the world frame (zero for PID)
        const V3T<T> v_ref = v3t<T>(fma_(m.cpsi, m.v_cmd.x, mul_(m.nspsi, m.v_cmd.y)), fma_(m.spsi, m.v_cmd.x, mul_(m.cpsi, m.v_cmd.y)), m.v_cmd.z);
        // position loop, Eq.9
        Ip.x = clamp_(fma_(m.e_p.x, P.dt_c, Ip.x), -P.int_clamp_pos, P.int_clamp_pos);
        Ip.y = clamp_(fma_(m.e_p.y, P.dt_c, Ip.y), -P.int_clamp_pos, P.int_clamp_pos);
        Ip.z = clamp_(fma_(m.e_p.z, P.dt_c, Ip.z), -P.int_clamp_pos, P.int_clamp_pos);
        const T ax = fma_(P.Kp_pos[0], m.e_p.x, fma_(P.Ki_pos[0], Ip.x, fma_(P.Kd_pos[0], sub_(v_ref.x, v.x), P.a_ff[0])));
        const T ay = fma_(P.Kp_pos[1], m.e_p.y, fma_(P.Ki_pos[1], Ip.y, fma_(P.Kd_pos[1], sub_(v_ref.y, v.y), P.a_ff[1])));
        const T az = add_(fma_(P.Kp_pos[2], m.e_p.z, fma_(P.Ki_pos[2], Ip.z, fma_(P.Kd_pos[2], sub_(v_ref.z, v.z), P.a_ff[2]))), P.g);
        thrust = clamp_(mul_(P.m, sqrt_(fma_(ax, ax, fma_(ay, ay, mul_(az, az))))), 0.0f, P.T_max);       // T = m |a*|
        phi_ref = clamp_(mul_(fma_(ax, m.spsi, mul_(ay, m.ncpsi)), P.inv_g), -P.tilt_max, P.tilt_max);    // small-angle tilt target
        th_ref = clamp_(mul_(fma_(ax, m.cpsi, mul_(ay, m.spsi)), P.inv_g), -P.tilt_max, P.tilt_max);
    }
    const V3T<T> e_eta = v3t<T>(sub_(phi_ref, m.roll), sub_(th_ref, m.pitch), m.e_psi);
    Ie.x = clamp_(fma_(e_eta.x, P.dt_c, Ie.x), -P.int_clamp_att, P.int_clamp_att);
    Ie.y = clamp_(fma_(e_eta.y, P.dt_c, Ie.y), -P.int_clamp_att, P.int_clamp_att);
    Ie.z = clamp_(fma_(e_eta.z, P.dt_c, Ie.z), -P.int_clamp_att, P.int_clamp_att);
    const T tx = clamp_(fma_(P.Kp_att[0], e_eta.x, fma_(P.Ki_att[0], Ie.x, mul_(-P.Kd_att[0], w.x))), -P.tau_xy_max, P.tau_xy_max);
    const T ty = clamp_(fma_(P.Kp_att[1], e_eta.y, fma_(P.Ki_att[1], Ie.y, mul_(-P.Kd_att[1], w.y))), -P.tau_xy_max, P.tau_xy_max);
    const T tz = clamp_(fma_(P.Kp_att[2], e_eta.z, fma_(P.Ki_att[2], Ie.z, mul_(-P.Kd_att[2], w.z))), -P.tau_z_max, P.tau_z_max);
    // closed-form allocation inverse, per-rotor clip, back to RPM.  (The clamps above are per-half min / max, so the products
    // below never sit next to a packed add: nothing for ptxas to contract differently in the two lane shapes.)
    T s0, s1, s2, s3;
    if (Feat<FEAT>::has(P, F_CF2P)) {     // +-configuration: tau_x = L (s1 - s3), tau_y = L (s2 - s0)
        const T qa = fma_(mul_(2.0f, tx), P.inv_arm, 0.0f), qb = fma_(mul_(2.0f, ty), P.inv_arm, 0.0f), qc = fma_(tz, P.inv_kappa, 0.0f);
        s0 = mul_(0.25f, sub_(sub_(thrust, qb), qc)); s1 = mul_(0.25f, add_(add_(thrust, qa), qc));
        s2 = mul_(0.25f, sub_(add_(thrust, qb), qc)); s3 = mul_(0.25f, add_(sub_(thrust, qa), qc));
    } else {
        const T qa = fma_(tx, P.inv_l, 0.0f), qb = fma_(ty, P.inv_l, 0.0f), qc = fma_(tz, P.inv_kappa, 0.0f);   // fma(a, b, 0): summed next (see ang_acc_t)
        s0 = mul_(0.25f, sub_(sub_(add_(thrust, qa), qb), qc)); s1 = mul_(0.25f, add_(add_(add_(thrust, qa), qb), qc));
        s2 = mul_(0.25f, sub_(add_(sub_(thrust, qa), qb), qc)); s3 = mul_(0.25f, add_(sub_(sub_(thrust, qa), qb), qc));
    }
    n[0] = sqrt_(mul_(clamp_(s0, 0.0f, P.s_max), P.inv_k_f)); n[1] = sqrt_(mul_(clamp_(s1, 0.0f, P.s_max), P.inv_k_f));
    n[2] = sqrt_(mul_(clamp_(s2, 0.0f, P.s_max), P.inv_k_f)); n[3] = sqrt_(mul_(clamp_(s3, 0.0f, P.s_max), P.inv_k_f));
}

// angular acceleration J^-1 (tau_body - w x J w); axisym: J_xx == J_yy, the z component has no gyroscopic term
__device__ __forceinline__ V3 ang_acc(const DevParams& P, V3 tb, V3 w, bool axisym) {
    return v3(fmaf(P.invJ[0], tb.x, -P.gyro[0] * (w.y * w.z)),
              fmaf(P.invJ[1], tb.y, -P.gyro[1] * (w.z * w.x)),
              axisym ? P.invJ[2] * tb.z : fmaf(P.invJ[2], tb.z, -P.gyro[2] * (w.x * w.y)));
}

// four standard normal values from one Philox draw: Box-Muller on (x, y) and on (z, w), the angle taken in [-pi, pi) so that
// the MUFU sine / cosine keep their accuracy (cos(a - pi) = -cos a is absorbed in the sign of the radius)
// The radius uses log1pf: MUFU.LG2's absolute error near 1 would show in the rare small radii (this path is optional, off the
// benchmark kernels' critical path).
__device__ __forceinline__ float4 normals4(uint4 r) {
    const float r1 = -fast_sqrt(-2.0f * log1pf(-u01(r.x))), r2 = -fast_sqrt(-2.0f * log1pf(-u01(r.z)));
    const float a1 = 6.28318531f * (u01(r.y) - 0.5f), a2 = 6.28318531f * (u01(r.w) - 0.5f);
    return make_float4(r1 * cos_fast(a1), r1 * sin_fast(a1), r2 * cos_fast(a2), r2 * sin_fast(a2));
}
// Table 4 sensor rows (reading Q49): what the observation emitted at step index t reports for
// [p, eta, v, omega] = the true value + sigma xi (xi fresh every step, streams 11..13) + beta b (b drawn at the reset
// index t - ep_step of the running episode, streams 14..16).  The twelve values follow the row order p, eta, v, omega.
struct Sensed { V3 p, eta, v, w; Q4 q; };                         // the kinematic entries as the observation reports them
__device__ __forceinline__ Sensed sensed(const DroneRegs& d, V3 eta) { Sensed s; s.p = d.p; s.eta = eta; s.v = d.v; s.w = d.w; s.q = d.q; return s; }
__device__ __forceinline__ void sense(const DevParams& P, unsigned e, uint32_t j, uint32_t t, uint32_t ep_step, Sensed& s) {
    const uint32_t eg = e + P.env_base, t0 = t - ep_step;
    // a set of standard deviations that is all zero multiplies its draws by zero: they are not made (warp-uniform branches;
    // 0 stands in for the normals, which leaves every sum below what it was)
    float4 n0 = make_float4(0.0f, 0.0f, 0.0f, 0.0f), n1 = n0, n2 = n0, b0 = n0, b1 = n0, b2 = n0;
    if (P.sens_mask & 1u) {
        n0 = normals4(philox4x32_10(eg, j, t, STREAM_OBS_NOISE, P.seed_lo, P.seed_hi));
        n1 = normals4(philox4x32_10(eg, j, t, STREAM_OBS_NOISE + 1, P.seed_lo, P.seed_hi));
        n2 = normals4(philox4x32_10(eg, j, t, STREAM_OBS_NOISE + 2, P.seed_lo, P.seed_hi));
    }
    if (P.sens_mask & 2u) {
        b0 = normals4(philox4x32_10(eg, j, t0, STREAM_OBS_BIAS, P.seed_lo, P.seed_hi));
        b1 = normals4(philox4x32_10(eg, j, t0, STREAM_OBS_BIAS + 1, P.seed_lo, P.seed_hi));
        b2 = normals4(philox4x32_10(eg, j, t0, STREAM_OBS_BIAS + 2, P.seed_lo, P.seed_hi));
    }
    const float sp = P.obs_noise[0], sv = P.obs_noise[1], se = P.obs_noise[2], sw = P.obs_noise[3];
    const float bp = P.obs_bias[0], bv = P.obs_bias[1], be = P.obs_bias[2], bw = P.obs_bias[3];
    s.p.x += fmaf(sp, n0.x, bp * b0.x); s.p.y += fmaf(sp, n0.y, bp * b0.y); s.p.z += fmaf(sp, n0.z, bp * b0.z);
    s.eta.x += fmaf(se, n0.w, be * b0.w); s.eta.y += fmaf(se, n1.x, be * b1.x); s.eta.z += fmaf(se, n1.y, be * b1.y);
    s.v.x += fmaf(sv, n1.z, bv * b1.z); s.v.y += fmaf(sv, n1.w, bv * b1.w); s.v.z += fmaf(sv, n2.x, bv * b2.x);
    s.w.x += fmaf(sw, n2.y, bw * b2.y); s.w.y += fmaf(sw, n2.z, bw * b2.z); s.w.z += fmaf(sw, n2.w, bw * b2.w);
}

// Observation row of one drone: [p, eta, v, w (, adjacency)] or KIN20 [p, q, eta, v, w, a], written as
// float4s when the row is 16 B aligned
template <int G>
__device__ __forceinline__ void write_obs(const DevParams& P, float* __restrict__ obs, size_t drone, const DroneRegs& d,
                                          const Sensed& s, const float (&adj)[G], int mode, float4 act, float4 tg) {
    const bool with_adj = mode == 1;
    float* o = obs + drone * (size_t)P.opd;
    if (mode == 2) {
        float4* o4 = reinterpret_cast<float4*>(o);                 // 20 floats per drone: always 16 B aligned
        o4[0] = make_float4(s.p.x, s.p.y, s.p.z, s.q.w);
        o4[1] = make_float4(s.q.x, s.q.y, s.q.z, s.eta.x);
        o4[2] = make_float4(s.eta.y, s.eta.z, s.v.x, s.v.y);
        o4[3] = make_float4(s.v.z, s.w.x, s.w.y, s.w.z);
        o4[4] = act;
        return;
    }
    if ((P.opd & 3) == 0) {
        float4* o4 = reinterpret_cast<float4*>(o);
        o4[0] = make_float4(s.p.x, s.p.y, s.p.z, s.eta.x);
        o4[1] = make_float4(s.eta.y, s.eta.z, s.v.x, s.v.y);
        o4[2] = make_float4(s.v.z, s.w.x, s.w.y, s.w.z);
        if (mode == 3) o4[3] = tg;                                 // KIN12_TGT
        if (with_adj) {
            if (G == 4) o4[3] = make_float4(adj[0], adj[1 % G], adj[2 % G], adj[3 % G]);
            else {
#pragma unroll
                for (int k = 0; k < G; ++k) if (k < P.M) o[12 + k] = adj[k];
            }
        }
    } else {
        o[0] = s.p.x; o[1] = s.p.y; o[2] = s.p.z; o[3] = s.eta.x; o[4] = s.eta.y; o[5] = s.eta.z;
        o[6] = s.v.x; o[7] = s.v.y; o[8] = s.v.z; o[9] = s.w.x; o[10] = s.w.y; o[11] = s.w.z;
        if (mode == 5) o[12] = tg.z;                               // KIN12_Z
        if (mode == 4) {                                           // KIN12_WP: next waypoint, world and body frame
            const V3 rb = rot_inv(d.q, v3(tg.x - d.p.x, tg.y - d.p.y, tg.z - d.p.z));
            o[12] = tg.x; o[13] = tg.y; o[14] = tg.z; o[15] = rb.x; o[16] = rb.y; o[17] = rb.z;
        }
        if (with_adj) {
#pragma unroll
            for (int k = 0; k < G; ++k) if (k < P.M) o[12 + k] = adj[k];
        }
    }
}

// adjacency row of this lane's drone: A_k = 1 if k == j or |p - p_k| < radius (Q23); whole-warp call
template <int G>
__device__ __forceinline__ void adjacency(const DevParams& P, V3 p, int lane, int j, float (&adj)[G]) {
    const unsigned mask = MDG_FULL;
    const int gbase = lane & ~(G - 1);
#pragma unroll
    for (int k = 0; k < G; ++k) {
        const float ox = __shfl_sync(mask, p.x, gbase + k), oy = __shfl_sync(mask, p.y, gbase + k),
                    oz = __shfl_sync(mask, p.z, gbase + k);
        const float dx = p.x - ox, dy = p.y - oy, dz = p.z - oz;
        adj[k] = (k == j || fmaf(dx, dx, fmaf(dy, dy, dz * dz)) < P.adj_radius2) ? 1.0f : 0.0f;
    }
}
template <int G> __device__ __forceinline__ float group_sum(float x) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) x += __shfl_xor_sync(MDG_FULL, x, o);
    return x;
}
template <int G> __device__ __forceinline__ int group_or(int x) {
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) x |= __shfl_xor_sync(MDG_FULL, x, o);
    return x;
}

}  // namespace mdg

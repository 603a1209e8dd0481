// mdg_dev.cuh — device-side parameter block, Philox4x32-10 and small fp32 helpers of the fused
// drone-env step kernel (sm_100a).  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mdg {

// Feature word of a kernel specialisation (compile-time when >= 0, read from DevParams when < 0).
enum : int {
    F_GND = 1, F_DRAG = 2, F_DW = 4, F_WIND = 8,          // == MDG_AERO_*
    F_EULER = 16,                                         // DYN integrator (Table 1)
    F_ACT_SHIFT = 5,                                      // 3 bits: MDG_ACT_*
    F_DSL = 1 << 8,
    F_OBS_SHIFT = 9,                                      // 3 bits: MDG_OBS_* (compare the field: Feat::obs)
    F_REW_SHIFT = 12,                                     // 3 bits: MDG_REW_*
    F_TERM_SHIFT = 15,                                    // 2 bits: MDG_TERM_*
    F_TGT_CIRCLE = 1 << 17,                               // targets are the formation circle slots (chord table)
    F_FULL = 1 << 18,                                     // n_drones == G: no padding lanes in a group
    F_AXISYM = 1 << 19,                                   // J_xx == J_yy: no gyroscopic term about body z
    F_CF2P = 1 << 20,                                     // +-configuration mixing
    F_DR = 1 << 21,                                       // per-episode domain-randomisation factors (Table 4)
    F_MLAG = 1 << 23,                                     // motor lag: rotor-speed state, wrench recomputed every substep
    F_SENS = 1 << 24,                                     // Table 4 sensor rows: noise / per-episode bias on the emitted observation
    F_LAT = 1 << 25,                                      // Table 4 latency rows: delayed action rows / sensed state (generic kernel)
    F_PATH = 1 << 26,                                     // formation centre on a closed polygonal path (generic kernel)
    F_WIND_MIX = 1 << 22,                                 // wind_mask != MDG_WIND_DRYDEN: only the generic kernel handles it
};

// Everything the kernels need, precomputed on the host in double and rounded once to fp32.
// Passed by value as a __grid_constant__ kernel parameter, so every field is a constant-bank operand.
struct DevParams {
    int N, M, K, ep_steps, auto_reset, feat;
    int reset_layout, target_mode, grid_cols, grid_rows, opd;
    uint32_t seed_lo, seed_hi, env_base;
    uint32_t static_items;                                // grid does not fill the device: one item per warp, item = warp index (no dispenser)
    uint32_t zero;                                        // always 0, unknown to the compiler (mdg_kernels.cuh: prefetch_item)
    uint32_t seq, chain;                                  // per launch: step sequence number, item-level chaining behind step seq - 1 (mdg_kernels.cuh)
    // integrator
    float h, half_h, h_sixth, half_h2, w2_exact[2];          // w2_exact: |omega|^2 above which the exact path runs
    // Rodrigues coefficients of R(c w)^T as polynomials in y = |w|^2, c = h/2 (stages 2, 3) and h (stage 4):
    // A(y) = c sin(c|w|)/(c|w|), B(y) = c^2 (1 - cos(c|w|))/(c|w|)^2.  Degree 2 (first three coefficients) is exact to
    // 1e-7 for |w| h <= 0.28 rad and is used where a controller keeps the body rates small (PID / VEL actions);
    // degree 3 holds to 0.75 rad and serves the open-loop action types.  w2_exact[d-2] is the matching |w|^2 bound.
    float rotA_half[4], rotB_half[4], rotA_full[4], rotB_full[4];
    float rotnA_half[4], rotnA_full[4], ngyro[3];            // -A's coefficients and -gyro: the lane-generic substep loop never negates
    // Eq.7 increment for phi = (h/6) s, s = w0 + 2 w2 + 2 w3 + w4, as polynomials in |s|^2: cos(|phi|/2) and (h/6) sin(|phi|/2)/|phi|
    float expC[4], expS[4], expCm[4], expSm[4];   // Eq.7 series for phi = (h/6) s and for phi = h s
    float inv_m, g, J[3], invJ[3], gyro[3];               // gyro = ((Jz-Jy)/Jx, (Jx-Jz)/Jy, (Jy-Jx)/Jz)
    // motor model (Eq.1-3)
    float k_f, inv_k_f, l, kappa, inv_l, inv_kappa, max_rpm, s_max, T_max, rpm2rad;
    float hover_rpm, rpm_span, arm, inv_arm;              // normalised-RPM map (HOVER, MAX - HOVER); arm length L for CF2P
    // aero (Eq.4-6) and wind
    float gnd_coef, h_clip, c_xy, c_z, dw_coef, dw_C2, dw_C3, dz_clip, inv_dz_clip;
    float dw_C2s, dw_C3s, dw_b2_min, dz_floor;            // Eq.6 with beta scaled by sqrt(2 ln 2): exp(-x/2b^2) = 2^(-x/b'^2)
    float wind_alpha, wind_gain, k_wind;
    float dryden_x, dryden_h_min, wind_sigma, inv_M;      // altitude-dependent Dryden scale: dt_c V (0 = fixed tau), altitude floor
    float gust_prob, gust_max, gust_ds;                   // MDG_WIND_GUST: trigger probability, largest speed, dt_c / duration
    int wind_mask; float wind_const[3], wind_sine_amp, wind_sine_omega;   // MDG_WIND_*: 1 AR(1) gust, 2 constant, 8 sinusoidal force
    // cascaded PID (Eq.9, Table 6)
    float dt_c, m, inv_g;
    float Kp_pos[3], Ki_pos[3], Kd_pos[3], Kp_att[3], Ki_att[3], Kd_att[3];
    float int_clamp_pos, int_clamp_att, pos_step_max, yaw_step_max, a_ff[3], tilt_max, tau_xy_max, tau_z_max;
    // epilogue
    float adj_radius2, at_target_radius2, term_tilt, term_dist2, term_center[3], z_max;   // radii squared
    // reset / targets
    float reset_center[3], reset_half[3], reset_z_lo, reset_z_hi, grid_spacing, circle_radius;
    float target_fixed[3], target_lo[3], target_hi[3], target_w_lo, target_w_hi, mh_z_lo, mh_z_hi, form_center[3], form_radius;
    int n_waypoints, wp_total; float waypoints[24], wp_radius2, wp_bonus, wp_shaping, wp_speed, wp_omega;   // waypoint tasks
    float dr_alpha[12];                                   // half-widths of the DR factors [m, J, k_f, k_m, drag, gnd, dw, g, motor, arm, max_rpm, -]
    float reset_rpy_half[3], reset_vel_half[3];           // Table 4 "init" row
    float motor_lag_lo, motor_lag_hi;                     // Table 4 motor lag: range of the time constant (s)
    int path_n; float path[24], path_len[8], path_perimeter, path_rate;   // moving formation centre: vertices, side lengths, form_speed dt_c
    int lat_a_lo, lat_a_n, lat_s_lo, lat_s_n;             // Table 4 latency rows in substeps: smallest delay and number of values (0 = off)
    float obs_noise[4], obs_bias[4];                      // Table 4 sensor rows: standard deviations for [position, velocity, RPY, body rates]
    unsigned sens_mask;                                   // bit 0: some obs_noise is non-zero, bit 1: some obs_bias (what is all zero is not drawn)
    float chord[32];                                      // distance between circle slots i and k: chord[|i - k|]
};

// SoA state planes (float4 per drone) and per-env words.  DESIGN.md §5.
struct DevBuffers {
    float4* P0;   // px py pz qw
    float4* P1;   // qx qy qz vx
    float4* P2;   // vy vz wx wy
    float4* P3;   // wz Ipx Ipy Ipz
    float4* P4;   // Iex Iey Iez -
    float4* P5;   // held setpoint x y z psi
    float4* P6;   // target x y z psi
    float4* R0;   // DR factors m J k_f k_m
    float4* R1;   // DR factors drag gnd dw g
    float4* R2;   // DR per-motor thrust bias
    float4* R3;   // DR arm, MAX_RPM, motor-lag time constant, -
    float4* N0;   // rotor speeds actually turning (motor lag state)
    float4* H0;   // action rows issued 1, 2 and 3 control steps ago (action latency; allocated only when it is on)
    float4* H1;
    float4* H2;
    float4* E0;   // wind x y z, bits(ep_step)
    float4* E1;   // running gust impulse: velocity x y z, progress s (>= 1: none)
    uint32_t* gstep;
    unsigned* ticket;   // [0..3] four work-item dispensers of the step kernel (0 between launches), used in turn
    unsigned* item_seq; // per work item: sequence number of the last step that finished it
    float* obs;
    float* reward;
    float* reward_d;   // [D] per-drone share of the reward
    uint8_t* done;
};

static const uint32_t STREAM_RESET_POS = 0, STREAM_RESET_EXTRA = 1, STREAM_WIND = 2, STREAM_ACTION = 3, STREAM_DR0 = 4, STREAM_DR1 = 5, STREAM_DR2 = 6, STREAM_DR3 = 7, STREAM_INIT_RPY = 8, STREAM_INIT_VEL = 9, STREAM_GUST = 10,
                      STREAM_OBS_NOISE = 11 /* 11..13 */, STREAM_OBS_BIAS = 14 /* 14..16 */, STREAM_LATENCY = 17;

// Philox4x32-10 (Salmon et al., SC'11).  key = seed halves, counter = (env, drone|~0, step, stream).
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}
__device__ __forceinline__ float u01(uint32_t x) { return (float)(x >> 8) * (1.0f / 16777216.0f); }

// MUFU approximations with flush-to-zero: a single SFU instruction each, no denormal rescaling code
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_fast(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float ex2_fast(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

__device__ __forceinline__ float lg2_fast(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sin_fast(float x) { float r; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float cos_fast(float x) { float r; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// atan2(y, x) to 2e-7 rad: octant reduction to a = min/max in [0, 1], a P(a^2) with a degree-7 minimax P
// (fitted for this kernel, max error 9e-8), one MUFU.RCP.  atan2(0, 0) = 0.
__device__ __forceinline__ float atan2_fast(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mx = fmaxf(fmaxf(ax, ay), 1e-30f), mn = fminf(ax, ay);
    const float a = mn * rcp_fast(mx), s = a * a;
    float p = fmaf(s, -4.780359644e-3f, 2.455679293e-2f);
    p = fmaf(s, p, -5.990426529e-2f); p = fmaf(s, p, 9.942728849e-2f); p = fmaf(s, p, -1.402940935e-1f);
    p = fmaf(s, p, 1.997137346e-1f); p = fmaf(s, p, -3.333209341e-1f); p = fmaf(s, p, 9.999999114e-1f);
    float r = a * p;
    r = ay > ax ? 1.57079632679f - r : r;
    r = x < 0.0f ? 3.14159265359f - r : r;
    return copysignf(r, y);
}
// asin(s) for |s| <= 1 to 1e-7: z + z t Q(t) on |s| <= 1/2 (t = s^2), pi/2 - 2 asin(sqrt((1 - |s|)/2)) above
__device__ __forceinline__ float asin_fast(float s) {
    const float a = fabsf(s);
    const bool big = a > 0.5f;
    const float t = big ? fmaf(-0.5f, a, 0.5f) : a * a;
    const float z = big ? t * rsqrt_fast(fmaxf(t, 1e-30f)) : a;
    float q = fmaf(t, 3.828223139e-2f, 2.645942860e-2f);
    q = fmaf(t, q, 4.501529088e-2f); q = fmaf(t, q, 7.498796169e-2f); q = fmaf(t, q, 1.666667248e-1f);
    const float r = fmaf(z * t, q, z);
    return copysignf(big ? fmaf(-2.0f, r, 1.57079632679f) : r, s);
}

struct V3 { float x, y, z; };
__device__ __forceinline__ V3 v3(float x, float y, float z) { V3 r; r.x = x; r.y = y; r.z = z; return r; }
__device__ __forceinline__ V3 cross(V3 a, V3 b) {
    return v3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
struct Q4 { float w, x, y, z; };

// rotate v by unit quaternion q (body -> world): v + w t + u x t, t = 2 u x v
__device__ __forceinline__ V3 rot(Q4 q, V3 v) {
    const V3 u = v3(q.x, q.y, q.z);
    const V3 t = cross(u, v);
    const V3 c = cross(u, t);
    return v3(fmaf(2.0f, fmaf(q.w, t.x, c.x), v.x), fmaf(2.0f, fmaf(q.w, t.y, c.y), v.y), fmaf(2.0f, fmaf(q.w, t.z, c.z), v.z));
}
// rotate v by the conjugate of q (world -> body)
__device__ __forceinline__ V3 rot_inv(Q4 q, V3 v) {
    Q4 c; c.w = q.w; c.x = -q.x; c.y = -q.y; c.z = -q.z;
    return rot(c, v);
}
__device__ __forceinline__ Q4 qmul(Q4 a, Q4 b) {
    Q4 r;
    r.w = a.w * b.w - a.x * b.x - a.y * b.y - a.z * b.z;
    r.x = a.w * b.x + b.w * a.x + (a.y * b.z - a.z * b.y);
    r.y = a.w * b.y + b.w * a.y + (a.z * b.x - a.x * b.z);
    r.z = a.w * b.z + b.w * a.z + (a.x * b.y - a.y * b.x);
    return r;
}
// Eq.7 increment: [cos(|phi|/2), sin(|phi|/2) phi/|phi|].  Both factors are even power series in
// x = |phi|^2, so no sqrt, division or MUFU is needed.  Degree 3 in x: truncation error < 1e-8 for
// |phi| <= 0.75 rad.  The caller routes |omega| h > 0.28 rad to the exact (library sin/cos) path.
__device__ __forceinline__ Q4 exp_half(V3 phi) {
    const float x = fmaf(phi.x, phi.x, fmaf(phi.y, phi.y, phi.z * phi.z));
    const float c = fmaf(x, fmaf(x, fmaf(x, -2.1701389e-5f, 2.6041667e-3f), -0.125f), 1.0f);
    const float s = fmaf(x, fmaf(x, fmaf(x, -1.5500992e-6f, 2.6041667e-4f), -2.0833333e-2f), 0.5f);
    Q4 r; r.w = c; r.x = s * phi.x; r.y = s * phi.y; r.z = s * phi.z;
    return r;
}
// the same increment for phi = c s with c folded into host-made coefficients (DevParams::expC, expS; degree 2 in |s|^2,
// error < 1e-8 for |phi| <= 0.28 rad; degree 3 for |phi| <= 0.75 rad)
template <int DEG>
__device__ __forceinline__ Q4 exp_half_scaled(const float (&cC)[4], const float (&cS)[4], V3 s) {
    const float y = fmaf(s.x, s.x, fmaf(s.y, s.y, s.z * s.z));
    const float c = DEG == 2 ? fmaf(y, fmaf(y, cC[2], cC[1]), cC[0]) : fmaf(y, fmaf(y, fmaf(y, cC[3], cC[2]), cC[1]), cC[0]);
    const float f = DEG == 2 ? fmaf(y, fmaf(y, cS[2], cS[1]), cS[0]) : fmaf(y, fmaf(y, fmaf(y, cS[3], cS[2]), cS[1]), cS[0]);
    Q4 r; r.w = c; r.x = f * s.x; r.y = f * s.y; r.z = f * s.z;
    return r;
}
__device__ __forceinline__ Q4 exp_half_exact(V3 phi) {
    const float x = fmaf(phi.x, phi.x, fmaf(phi.y, phi.y, phi.z * phi.z));
    if (x <= 0.07f) return exp_half(phi);
    const float n = sqrtf(x);
    float sn, cn;
    sincosf(0.5f * n, &sn, &cn);
    const float s = sn / n;
    Q4 r; r.w = cn; r.x = s * phi.x; r.y = s * phi.y; r.z = s * phi.z;
    return r;
}
// R(c w)^T tau for the rotation vector phi = c w (Rodrigues): tau - A(y) (w x tau) + B(y) w x (w x tau) with
// y = |w|^2 and the step factor c folded into the host-made coefficients cA, cB (DevParams::rotA_*, rotB_*;
// degree 2 in y: error < 1e-7 relative for c|w| <= 0.28 rad; degree 3: for c|w| <= 0.75 rad).  Used for the RK4 stage torques.
template <int DEG>
__device__ __forceinline__ V3 stage_torque(const float (&cA)[4], const float (&cB)[4], V3 w, V3 tau) {
    const float y = fmaf(w.x, w.x, fmaf(w.y, w.y, w.z * w.z));
    const float A = DEG == 2 ? fmaf(y, fmaf(y, cA[2], cA[1]), cA[0]) : fmaf(y, fmaf(y, fmaf(y, cA[3], cA[2]), cA[1]), cA[0]);
    const float Bc = DEG == 2 ? fmaf(y, fmaf(y, cB[2], cB[1]), cB[0]) : fmaf(y, fmaf(y, fmaf(y, cB[3], cB[2]), cB[1]), cB[0]);
    const V3 c1 = cross(w, tau);
    const V3 c2 = cross(w, c1);
    return v3(fmaf(Bc, c2.x, fmaf(-A, c1.x, tau.x)), fmaf(Bc, c2.y, fmaf(-A, c1.y, tau.y)), fmaf(Bc, c2.z, fmaf(-A, c1.z, tau.z)));
}
// ---- lane-generic arithmetic of the substep loop ----------------------------------------------------------------------
// The substep loop is written once over a value type T: float (one drone per thread) or F2, a pair of floats in one 64-bit
// register holding the same quantity of TWO drones (two envs per lane group).  sm_100 executes fma / mul / add on such pairs
// as single instructions (FFMA2 / FMUL2 / FADD2: one issue slot, two cycles of the FP32 pipe), which is what an issue-bound
// kernel needs; everything else (MUFU, min / max, compares, selects, shuffles) works on the halves, which are ordinary
// registers.  Every operation is spelled out (no operator the compiler could contract differently), so both instantiations
// round identically: the two-drones-per-thread kernel is bit for bit the one-drone kernel.
struct F2 { unsigned long long v; };
__device__ __forceinline__ F2 pk(float lo, float hi) { F2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo_(F2 a) { float l, h; asm("mov.b64 {%0, %1}, %2;" : "=f"(l), "=f"(h) : "l"(a.v)); return l; }
__device__ __forceinline__ float hi_(F2 a) { float l, h; asm("mov.b64 {%0, %1}, %2;" : "=f"(l), "=f"(h) : "l"(a.v)); return h; }
struct B2 { bool lo, hi; };
template <class T> struct LaneOps;
template <> struct LaneOps<float> {
    typedef bool mask;
    static __device__ __forceinline__ float bc(float s) { return s; }
};
template <> struct LaneOps<F2> {
    typedef B2 mask;
    static __device__ __forceinline__ F2 bc(float s) { return pk(s, s); }
};
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float mul_(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float neg_(float a) { return -a; }
__device__ __forceinline__ F2 fma_(F2 a, F2 b, F2 c) { F2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
__device__ __forceinline__ F2 mul_(F2 a, F2 b) { F2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ F2 add_(F2 a, F2 b) { F2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ F2 sub_(F2 a, F2 b) { F2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ F2 neg_(F2 a) { F2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(0xBF800000BF800000ull)); return r; }   // x * -1: exact, one FMUL2 (two sign flips on the ALU pipe measured slower)
// uniform (float) operands broadcast to both halves
__device__ __forceinline__ F2 fma_(float a, F2 b, F2 c) { return fma_(pk(a, a), b, c); }
__device__ __forceinline__ F2 fma_(F2 a, float b, F2 c) { return fma_(a, pk(b, b), c); }
__device__ __forceinline__ F2 fma_(F2 a, F2 b, float c) { return fma_(a, b, pk(c, c)); }
__device__ __forceinline__ F2 fma_(float a, F2 b, float c) { return fma_(pk(a, a), b, pk(c, c)); }
__device__ __forceinline__ F2 fma_(F2 a, float b, float c) { return fma_(a, pk(b, b), pk(c, c)); }
__device__ __forceinline__ F2 mul_(float a, F2 b) { return mul_(pk(a, a), b); }
__device__ __forceinline__ F2 mul_(F2 a, float b) { return mul_(a, pk(b, b)); }
// per-half operations
#define MDG_MAP1(name, expr) \
    __device__ __forceinline__ float name(float x) { return expr; } \
    __device__ __forceinline__ F2 name(F2 a) { float x = lo_(a); const float l = expr; x = hi_(a); const float h = expr; return pk(l, h); }
MDG_MAP1(rcp_, rcp_fast(x))
MDG_MAP1(rsqrt_, rsqrt_fast(x))
MDG_MAP1(ex2n_, ex2_fast(-x))
MDG_MAP1(abs_, fabsf(x))
MDG_MAP1(sat_, __saturatef(x))
#undef MDG_MAP1
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ F2 max_(F2 a, float b) { return pk(fmaxf(lo_(a), b), fmaxf(hi_(a), b)); }
__device__ __forceinline__ bool gt_(float a, float b) { return a > b; }
__device__ __forceinline__ bool lt_(float a, float b) { return a < b; }
__device__ __forceinline__ B2 gt_(F2 a, float b) { B2 m; m.lo = lo_(a) > b; m.hi = hi_(a) > b; return m; }
__device__ __forceinline__ B2 lt_(F2 a, float b) { B2 m; m.lo = lo_(a) < b; m.hi = hi_(a) < b; return m; }
__device__ __forceinline__ bool and_(bool a, bool b) { return a && b; }
__device__ __forceinline__ B2 and_(B2 a, bool b) { B2 m; m.lo = a.lo && b; m.hi = a.hi && b; return m; }
__device__ __forceinline__ float sel_(bool m, float a, float b) { return m ? a : b; }
__device__ __forceinline__ F2 sel_(B2 m, F2 a, F2 b) { return pk(m.lo ? lo_(a) : lo_(b), m.hi ? hi_(a) : hi_(b)); }
__device__ __forceinline__ F2 sel_(B2 m, F2 a, float b) { return pk(m.lo ? lo_(a) : b, m.hi ? hi_(a) : b); }
__device__ __forceinline__ F2 sel_(B2 m, float a, F2 b) { return pk(m.lo ? a : lo_(b), m.hi ? a : hi_(b)); }
__device__ __forceinline__ float shfl_(float x, int src, int width) { return __shfl_sync(0xffffffffu, x, src, width); }
__device__ __forceinline__ F2 shfl_(F2 a, int src, int width) { return pk(__shfl_sync(0xffffffffu, lo_(a), src, width), __shfl_sync(0xffffffffu, hi_(a), src, width)); }

template <class T> struct V3T { T x, y, z; };
template <class T> struct Q4T { T w, x, y, z; };
template <class T> __device__ __forceinline__ V3T<T> v3t(T x, T y, T z) { V3T<T> r; r.x = x; r.y = y; r.z = z; return r; }
template <class T> __device__ __forceinline__ V3T<T> neg3(V3T<T> a) { return v3t<T>(neg_(a.x), neg_(a.y), neg_(a.z)); }
// a x b, given na = -a: each component is one multiply and one fma
template <class T> __device__ __forceinline__ V3T<T> cross_n(V3T<T> a, V3T<T> na, V3T<T> b) {
    return v3t<T>(fma_(a.y, b.z, mul_(na.z, b.y)), fma_(a.z, b.x, mul_(na.x, b.z)), fma_(a.x, b.y, mul_(na.y, b.x)));
}
template <class T> __device__ __forceinline__ T dot3(V3T<T> a, V3T<T> b) { return fma_(a.x, b.x, fma_(a.y, b.y, mul_(a.z, b.z))); }
// a (x) b (Hamilton product)
template <class T> __device__ __forceinline__ Q4T<T> qmul_t(Q4T<T> a, Q4T<T> b) {
    const T nx = neg_(a.x), ny = neg_(a.y), nz = neg_(a.z);
    Q4T<T> r;
    r.w = fma_(nz, b.z, fma_(ny, b.y, fma_(nx, b.x, mul_(a.w, b.w))));
    r.x = fma_(a.w, b.x, fma_(b.w, a.x, fma_(a.y, b.z, mul_(nz, b.y))));
    r.y = fma_(a.w, b.y, fma_(b.w, a.y, fma_(a.z, b.x, mul_(nx, b.z))));
    r.z = fma_(a.w, b.z, fma_(b.w, a.z, fma_(a.x, b.y, mul_(ny, b.x))));
    return r;
}
// polynomial c0 + y (c1 + y (c2 [+ y c3])) with uniform coefficients
template <int DEG, class T> __device__ __forceinline__ T poly_(const float (&c)[4], T y) {
    return DEG == 2 ? fma_(y, fma_(y, c[2], c[1]), c[0]) : fma_(y, fma_(y, fma_(y, c[3], c[2]), c[1]), c[0]);
}
// Eq.7 increment [cos(|phi|/2), sin(|phi|/2) phi/|phi|] for phi = c s with c folded into host-made coefficients (DevParams::expC, expS)
template <int DEG, class T> __device__ __forceinline__ Q4T<T> exp_half_scaled_t(const float (&cC)[4], const float (&cS)[4], V3T<T> s) {
    const T y = dot3(s, s);
    const T f = poly_<DEG>(cS, y);
    Q4T<T> r; r.w = poly_<DEG>(cC, y); r.x = mul_(f, s.x); r.y = mul_(f, s.y); r.z = mul_(f, s.z);
    return r;
}
// the same increment for an explicit rotation vector phi (degree 3, |phi| <= 0.75 rad): the DYN integrator's update
template <class T> __device__ __forceinline__ Q4T<T> exp_half_t(V3T<T> phi) {
    const T x = dot3(phi, phi);
    const T c = fma_(x, fma_(x, fma_(x, -2.1701389e-5f, 2.6041667e-3f), -0.125f), 1.0f);
    const T f = fma_(x, fma_(x, fma_(x, -1.5500992e-6f, 2.6041667e-4f), -2.0833333e-2f), 0.5f);
    Q4T<T> r; r.w = c; r.x = mul_(f, phi.x); r.y = mul_(f, phi.y); r.z = mul_(f, phi.z);
    return r;
}
// R(c w)^T tau for the rotation vector phi = c w (Rodrigues): tau - A(y) (w x tau) + B(y) w x (w x tau), y = |w|^2, the step
// factor c folded into the host-made coefficients; cnA holds -A's coefficients so that no negation is needed
template <int DEG, class T> __device__ __forceinline__ V3T<T> stage_torque_t(const float (&cnA)[4], const float (&cB)[4], V3T<T> w, V3T<T> tau) {
    const T y = dot3(w, w);
    const T nA = poly_<DEG>(cnA, y), Bc = poly_<DEG>(cB, y);
    const V3T<T> nw = neg3(w);
    const V3T<T> c1 = cross_n(w, nw, tau);
    const V3T<T> c2 = cross_n(w, nw, c1);
    return v3t<T>(fma_(Bc, c2.x, fma_(nA, c1.x, tau.x)), fma_(Bc, c2.y, fma_(nA, c1.y, tau.y)), fma_(Bc, c2.z, fma_(nA, c1.z, tau.z)));
}

// sqrt(x) for x >= 0: one MUFU.SQRT (sqrt.approx.ftz, 1 ulp; sqrt(0) = 0)
__device__ __forceinline__ float fast_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ F2 add_(F2 a, float b) { return add_(a, pk(b, b)); }
__device__ __forceinline__ float clamp_(float x, float lo, float hi) { return fminf(fmaxf(x, lo), hi); }
__device__ __forceinline__ F2 clamp_(F2 a, float lo, float hi) { return pk(fminf(fmaxf(lo_(a), lo), hi), fminf(fmaxf(hi_(a), lo), hi)); }
__device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ F2 min_(F2 a, F2 b) { return pk(fminf(lo_(a), lo_(b)), fminf(hi_(a), hi_(b))); }
__device__ __forceinline__ float sqrt_(float x) { return fast_sqrt(x); }
__device__ __forceinline__ F2 sqrt_(F2 a) { return pk(fast_sqrt(lo_(a)), fast_sqrt(hi_(a))); }
__device__ __forceinline__ float clampf(float x, float lo, float hi) { return fminf(fmaxf(x, lo), hi); }
__device__ __forceinline__ float wrap_pi(float x) {
    const float k = ceilf((x - 3.14159265358979f) * 0.159154943091895f);
    return fmaf(-6.28318530717959f, k, x);
}
// ZYX Euler angles (roll, pitch, yaw) of q
__device__ __forceinline__ float roll_of(Q4 q) { return atan2_fast(2.0f * fmaf(q.w, q.x, q.y * q.z), fmaf(-2.0f, fmaf(q.x, q.x, q.y * q.y), 1.0f)); }
__device__ __forceinline__ float pitch_of(Q4 q) { return asin_fast(clampf(2.0f * fmaf(q.w, q.y, -q.z * q.x), -1.0f, 1.0f)); }
__device__ __forceinline__ V3 euler_zyx(Q4 q) {
    V3 e;
    e.x = roll_of(q);
    e.y = pitch_of(q);
    e.z = atan2_fast(2.0f * fmaf(q.w, q.z, q.x * q.y), fmaf(-2.0f, fmaf(q.y, q.y, q.z * q.z), 1.0f));
    return e;
}

}  // namespace mdg

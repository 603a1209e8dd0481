// mdg_kernels.cuh — __global__ entry points: fused step, reset, obs refresh, harness action generator.
#pragma once
#include "mdg_step.cuh"

namespace mdg {

__device__ __forceinline__ void load_state(const DevBuffers& B, size_t d, DroneRegs& r) {
    const float4 a = B.P0[d], b = B.P1[d], c = B.P2[d], e = B.P3[d];
    r.p = v3(a.x, a.y, a.z); r.q.w = a.w; r.q.x = b.x; r.q.y = b.y; r.q.z = b.z;
    r.v = v3(b.w, c.x, c.y); r.w = v3(c.z, c.w, e.x); r.Ip = v3(e.y, e.z, e.w);
}
__device__ __forceinline__ void store_state(const DevBuffers& B, size_t d, const DroneRegs& r) {
    B.P0[d] = make_float4(r.p.x, r.p.y, r.p.z, r.q.w);
    B.P1[d] = make_float4(r.q.x, r.q.y, r.q.z, r.v.x);
    B.P2[d] = make_float4(r.v.y, r.v.z, r.w.x, r.w.y);
    B.P3[d] = make_float4(r.w.z, r.Ip.x, r.Ip.y, r.Ip.z);
}

// S8 rotation: classical RK4 on (q, w_body) with the torque frozen in the world frame (MJC* modes) or
// explicit Euler (DYN).  The stage orientation is q0 (x) dq, so the body-frame torque at a stage is
// R(dq)^T tau_b and q0 itself is only needed for the final update.  EXACT selects the library
// sin/cos for |omega| h > 2 rad; the hot path uses the branch-free series of exp_half.
template <bool EXACT, bool EULER>
__device__ __forceinline__ void integrate_rot(const DevParams& P, Q4& q, V3& w, V3 tau_b, V3 k1_tau) {
    auto ex = [](V3 phi) { return EXACT ? exp_half_exact(phi) : exp_half(phi); };
    if (!EULER) {
        const V3 w0 = w;
        const V3 k1 = v3(fmaf(-P.gyro[0], w0.y * w0.z, k1_tau.x), fmaf(-P.gyro[1], w0.z * w0.x, k1_tau.y),
                         fmaf(-P.gyro[2], w0.x * w0.y, k1_tau.z));
        const V3 w2 = v3(fmaf(P.half_h, k1.x, w0.x), fmaf(P.half_h, k1.y, w0.y), fmaf(P.half_h, k1.z, w0.z));
        auto stage = [&](V3 phi) { return EXACT ? rot_inv(exp_half_exact(phi), tau_b) : rotvec_inv(phi, tau_b); };
        const V3 k2 = ang_acc(P, stage(v3(P.half_h * w0.x, P.half_h * w0.y, P.half_h * w0.z)), w2);
        const V3 w3 = v3(fmaf(P.half_h, k2.x, w0.x), fmaf(P.half_h, k2.y, w0.y), fmaf(P.half_h, k2.z, w0.z));
        const V3 k3 = ang_acc(P, stage(v3(P.half_h * w2.x, P.half_h * w2.y, P.half_h * w2.z)), w3);
        const V3 w4 = v3(fmaf(P.h, k3.x, w0.x), fmaf(P.h, k3.y, w0.y), fmaf(P.h, k3.z, w0.z));
        const V3 k4 = ang_acc(P, stage(v3(P.h * w3.x, P.h * w3.y, P.h * w3.z)), w4);
        const V3 phi = v3(P.h_sixth * (w0.x + 2.0f * (w2.x + w3.x) + w4.x), P.h_sixth * (w0.y + 2.0f * (w2.y + w3.y) + w4.y),
                          P.h_sixth * (w0.z + 2.0f * (w2.z + w3.z) + w4.z));
        q = qmul(q, ex(phi));
        w = v3(fmaf(P.h_sixth, k1.x + 2.0f * (k2.x + k3.x) + k4.x, w0.x), fmaf(P.h_sixth, k1.y + 2.0f * (k2.y + k3.y) + k4.y, w0.y),
               fmaf(P.h_sixth, k1.z + 2.0f * (k2.z + k3.z) + k4.z, w0.z));
    } else {
        const V3 k1 = ang_acc(P, tau_b, w);
        w = v3(fmaf(P.h, k1.x, w.x), fmaf(P.h, k1.y, w.y), fmaf(P.h, k1.z, w.z));
        q = qmul(q, ex(v3(P.h * w.x, P.h * w.y, P.h * w.z)));
    }
    const float rn = rsqrt_fast(fmaf(q.w, q.w, fmaf(q.x, q.x, fmaf(q.y, q.y, q.z * q.z))));
    q.w *= rn; q.x *= rn; q.y *= rn; q.z *= rn;
}
// out-of-line copy for fast spins (|omega| h > 2 rad): rare, keeps the hot loop free of library calls
struct RotState { Q4 q; V3 w; };
template <bool EULER>
__device__ __noinline__ RotState integrate_rot_exact(const DevParams& P, Q4 q, V3 w, V3 tau_b, V3 k1_tau) {
    integrate_rot<true, EULER>(P, q, w, tau_b, k1_tau);
    RotState r; r.q = q; r.w = w;
    return r;
}

// One control step of every env.  Thread -> (env e, lane-in-group j).
// MINB = resident blocks of 128 threads per SM the register allocation must allow.
template <int G, int FEAT, int MINB>
__global__ void __launch_bounds__(128, MINB) step_kernel(const __grid_constant__ DevParams P, const DevBuffers B,
                                                         const float4* __restrict__ actions) {
    using F = Feat<FEAT>;
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned e_raw = tid / G;
    const int j = tid % G;
    const bool env_ok = e_raw < (unsigned)P.N;
    const unsigned e = env_ok ? e_raw : (unsigned)P.N - 1;      // idle lanes shadow the last env (no stores)
    const bool active = env_ok && j < P.M;
    const int jj = j < P.M ? j : P.M - 1;
    const size_t drone = (size_t)e * P.M + jj;
    const bool pid = F::act(P) != 0;

    DroneRegs d;
    load_state(B, drone, d);
    if (pid) {
        const float4 i4 = B.P4[drone];
        d.Ie = v3(i4.x, i4.y, i4.z);
        if (F::act(P) == 1) d.sp = B.P5[drone];
    }
    const float4 act4 = actions[drone];
    float4 env4 = B.E0[e];
    const uint32_t t = B.gstep[e] + 1u;

    // S7 wind gust: one AR(1) update per env and control step, force held over the substeps
    V3 Fwind = v3(0, 0, 0);
    if (F::has(P, F_WIND)) {
        const uint4 r = philox4x32_10(e + P.env_base, 0xFFFFFFFFu, t, STREAM_WIND, P.seed_lo, P.seed_hi);
        const float r1 = sqrtf(-2.0f * logf(1.0f - u01(r.x))), r2 = sqrtf(-2.0f * logf(1.0f - u01(r.z)));
        float s1, c1, s2, c2;
        sincospif(2.0f * u01(r.y), &s1, &c1);
        sincospif(2.0f * u01(r.w), &s2, &c2);
        env4.x = fmaf(P.wind_alpha, env4.x, P.wind_gain * (r1 * c1));
        env4.y = fmaf(P.wind_alpha, env4.y, P.wind_gain * (r1 * s1));
        env4.z = fmaf(P.wind_alpha, env4.z, P.wind_gain * (r2 * c2));
        const V3 rel = v3(env4.x - d.v.x, env4.y - d.v.y, env4.z - d.v.z);
        const float kn = P.k_wind * sqrtf(fmaf(rel.x, rel.x, fmaf(rel.y, rel.y, rel.z * rel.z)));
        Fwind = v3(kn * rel.x, kn * rel.y, kn * rel.z);
    }

    // S1/S2 decode, S3 motor model (Eq.1-3); RPMs are held over the K substeps
    float n[4];
    decode_action<FEAT>(P, act4, d, n);
    const float f0 = P.k_f * (n[0] * n[0]), f1 = P.k_f * (n[1] * n[1]), f2 = P.k_f * (n[2] * n[2]), f3 = P.k_f * (n[3] * n[3]);
    const float T = (f0 + f1) + (f2 + f3);
    const V3 tau_b = v3(P.l * ((f0 + f1) - (f2 + f3)), P.l * ((f1 + f2) - (f0 + f3)), P.kappa * ((f1 + f3) - (f0 + f2)));
    const float Om = P.rpm2rad * ((n[0] + n[1]) + (n[2] + n[3]));
    const V3 k1_tau = v3(P.invJ[0] * tau_b.x, P.invJ[1] * tau_b.y, P.invJ[2] * tau_b.z);
    const float cxy = -P.c_xy * Om, cz = -P.c_z * Om, gndT = P.gnd_coef * T;
    const float w2_slow = 1.0f / (P.h * P.h);                     // |omega| h > 1 rad
    const float dcz = cz - cxy;
    const bool full_group = P.M == G;

    bool hit = false;
#pragma unroll 1
    for (int k = 0; k < P.K; ++k) {
        // S4-S7 world-frame force from the start-of-substep state
        // b = R(q) z: thrust is T b, and Eq.5's R diag(c_xy, c_xy, c_z) R^T v = c_xy v + (c_z - c_xy)(b.v) b
        const V3 b = v3(2.0f * fmaf(d.q.x, d.q.z, d.q.w * d.q.y), 2.0f * fmaf(d.q.y, d.q.z, -d.q.w * d.q.x),
                        fmaf(-2.0f, fmaf(d.q.x, d.q.x, d.q.y * d.q.y), 1.0f));
        V3 Fw;
        if (F::has(P, F_DRAG)) {
            const float s = fmaf(dcz, fmaf(b.x, d.v.x, fmaf(b.y, d.v.y, b.z * d.v.z)), T);
            Fw = v3(fmaf(s, b.x, cxy * d.v.x), fmaf(s, b.y, cxy * d.v.y), fmaf(s, b.z, cxy * d.v.z));
        } else Fw = v3(T * b.x, T * b.y, T * b.z);
        if (F::has(P, F_GND)) {                                   // Eq.4, gated on body z pointing up
            const float r22 = b.z;
            const float hgt = fmaxf(d.p.z, P.h_clip);
            const float gain = gndT * rcp_fast(hgt * hgt);
            Fw.z += r22 > 0.0f ? gain : 0.0f;
        }
        if (G > 1 && F::has(P, F_DW)) {                           // Eq.6 over every drone above this one
            float dw = 0.0f;
#pragma unroll
            for (int kk = 1; kk < G; ++kk) {                      // partner lane = lane ^ kk: every other drone once
                const float ox = __shfl_xor_sync(MDG_FULL, d.p.x, kk), oy = __shfl_xor_sync(MDG_FULL, d.p.y, kk),
                            oz = __shfl_xor_sync(MDG_FULL, d.p.z, kk);
                const float dz = oz - d.p.z, dx = ox - d.p.x, dy = oy - d.p.y;
                const float dxy2 = fmaf(dx, dx, dy * dy);
                const float dze = fmaxf(dz, P.dz_clip);
                const float ramp = P.dz_clip > 0.0f ? fminf(dz * P.inv_dz_clip, 1.0f) : 1.0f;
                const float beta = fmaf(P.dw_C2, dze, P.dw_C3);
                const float b2 = beta * beta, z2 = dze * dze;
                const float rinv = rcp_fast(z2 * b2);                      // one reciprocal serves alpha and the exponent
                const float alpha = P.dw_coef * (b2 * rinv);
                const float ex = b2 < 1e-12f ? (dxy2 == 0.0f ? 1.0f : 0.0f) : ex2_fast(-0.72134752f * dxy2 * (z2 * rinv));   // exp(-x/2) = 2^(-x log2(e)/2)
                const float al = b2 < 1e-12f ? P.dw_coef * rcp_fast(z2) : alpha;
                const bool on = (full_group || (j ^ kk) < P.M) && dz > 0.0f && dxy2 < 100.0f;
                dw += on ? ramp * al * ex : 0.0f;
            }
            Fw.z -= dw;
        }
        if (F::has(P, F_WIND)) { Fw.x += Fwind.x; Fw.y += Fwind.y; Fw.z += Fwind.z; }
        const V3 acc = v3(Fw.x * P.inv_m, Fw.y * P.inv_m, fmaf(Fw.z, P.inv_m, -P.g));

        // S8 integrate with the wrench frozen in the world frame
        const bool fast_spin = fmaf(d.w.x, d.w.x, fmaf(d.w.y, d.w.y, d.w.z * d.w.z)) > w2_slow;
        if (!F::has(P, F_EULER)) {
            d.p.x = fmaf(P.half_h2, acc.x, fmaf(P.h, d.v.x, d.p.x));
            d.p.y = fmaf(P.half_h2, acc.y, fmaf(P.h, d.v.y, d.p.y));
            d.p.z = fmaf(P.half_h2, acc.z, fmaf(P.h, d.v.z, d.p.z));
            d.v.x = fmaf(P.h, acc.x, d.v.x); d.v.y = fmaf(P.h, acc.y, d.v.y); d.v.z = fmaf(P.h, acc.z, d.v.z);
            if (fast_spin) { const RotState rs = integrate_rot_exact<false>(P, d.q, d.w, tau_b, k1_tau); d.q = rs.q; d.w = rs.w; }
            else integrate_rot<false, false>(P, d.q, d.w, tau_b, k1_tau);
        } else {                                                   // DYN: explicit Euler
            d.v.x = fmaf(P.h, acc.x, d.v.x); d.v.y = fmaf(P.h, acc.y, d.v.y); d.v.z = fmaf(P.h, acc.z, d.v.z);
            d.p.x = fmaf(P.h, d.v.x, d.p.x); d.p.y = fmaf(P.h, d.v.y, d.p.y); d.p.z = fmaf(P.h, d.v.z, d.p.z);
            if (fast_spin) { const RotState rs = integrate_rot_exact<true>(P, d.q, d.w, tau_b, k1_tau); d.q = rs.q; d.w = rs.w; }
            else integrate_rot<false, true>(P, d.q, d.w, tau_b, k1_tau);
        }
        if (d.p.z < 0.0f) { hit = true; d.p.z = 0.0f; d.v.z = fmaxf(d.v.z, 0.0f); }   // floor
    }

    // S9-S11 epilogue on the end-of-step state
    const int lane = threadIdx.x & 31;
    const int gbase = lane & ~(G - 1);
    const float4 tg = B.P6[drone];
    V3 eta = euler_zyx(d.q);
    const int term = F::term(P);
    const float aphi = fabsf(eta.x), ath = fabsf(eta.y);
    int flags = 0;                                                 // bit0 terminated, bit1 crash
    if (term == 1 || term == 3) { if (hit) flags |= 3; if (d.p.z > P.z_max) flags |= 1; }
    if (term != 0 && (aphi > P.term_tilt || ath > P.term_tilt)) flags |= 3;
    if (term == 2 || term == 3) {
        const float dx = d.p.x - P.term_center[0], dy = d.p.y - P.term_center[1], dz = d.p.z - P.term_center[2];
        if (fmaf(dx, dx, fmaf(dy, dy, dz * dz)) > P.term_dist2) flags |= 1;
    }
    const float ex = d.p.x - tg.x, ey = d.p.y - tg.y, ez = d.p.z - tg.z;
    const float e2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
    float r;
    const int rew = F::rew(P);
    if (rew == 0 || rew == 2) {                                    // Eq.8, summed over drones
        const float speed = fast_sqrt(fmaf(d.v.x, d.v.x, fmaf(d.v.y, d.v.y, d.v.z * d.v.z)));
        r = -fabsf(ez) - 0.1f * fast_sqrt(fmaf(ex, ex, ey * ey)) - 0.05f * speed - 0.05f * (aphi + ath);
        if (e2 < P.at_target_radius2) r += 0.5f;
        if (flags & 2) r -= 100.0f;
    } else if (rew == 1) {
        r = -e2;
    } else {                                                       // formation: pair term below
        r = -fast_sqrt(e2);
    }
    if (G > 1 && rew == 3) {
        float pen = 0.0f;                                          // the self term is |0 - 0| = 0
#pragma unroll
        for (int kk = 0; kk < G; ++kk) {
            const float ox = __shfl_sync(MDG_FULL, d.p.x, gbase + kk), oy = __shfl_sync(MDG_FULL, d.p.y, gbase + kk),
                        oz = __shfl_sync(MDG_FULL, d.p.z, gbase + kk);
            const float ux = __shfl_sync(MDG_FULL, tg.x, gbase + kk), uy = __shfl_sync(MDG_FULL, tg.y, gbase + kk),
                        uz = __shfl_sync(MDG_FULL, tg.z, gbase + kk);
            const float ax = d.p.x - ox, ay = d.p.y - oy, az = d.p.z - oz;
            const float bx = tg.x - ux, by = tg.y - uy, bz = tg.z - uz;
            const float dact = fast_sqrt(fmaf(ax, ax, fmaf(ay, ay, az * az))), ddes = fast_sqrt(fmaf(bx, bx, fmaf(by, by, bz * bz)));
            pen += (full_group || kk < P.M) ? fabsf(dact - ddes) : 0.0f;
        }
        r = fmaf(-0.25f, pen, r);                                  // each unordered pair is seen from both ends
    }
    const float rsum = group_sum<G>(j < P.M ? r : 0.0f);
    const int gflags = group_or<G>(j < P.M ? flags : 0);
    const uint32_t ep = __float_as_uint(env4.w) + 1u;
    const bool truncated = P.ep_steps > 0 && (int)ep >= P.ep_steps;
    const int done = (gflags & 1) | (truncated ? 2 : 0);
    uint32_t ep_out = ep;
    float4 tg_out = tg;
    const bool do_reset = done != 0 && P.auto_reset != 0;
    if (do_reset) {                                                // S12 same-call auto-reset
        reset_drone(P, e, (uint32_t)jj, t, d, tg_out);
        env4.x = env4.y = env4.z = 0.0f; ep_out = 0u;
        eta = v3(0, 0, 0);
    }
    float adj[G];
#pragma unroll
    for (int kk = 0; kk < G; ++kk) adj[kk] = 0.0f;
    if (F::has(P, F_ADJ)) adjacency<G>(P, d.p, lane, j, adj);
    if (!active) return;
    store_state(B, drone, d);
    if (pid) {
        B.P4[drone] = make_float4(d.Ie.x, d.Ie.y, d.Ie.z, 0.0f);
        if (F::act(P) == 1) B.P5[drone] = d.sp;
    }
    if (do_reset) B.P6[drone] = tg_out;
    write_obs<G>(P, B.obs, drone, d, eta, adj, F::has(P, F_ADJ));
    if (j == 0) {
        env4.w = __uint_as_float(ep_out);
        B.E0[e] = env4; B.gstep[e] = t;
        B.reward[e] = rsum; B.done[e] = (uint8_t)done;
    }
}

// mdg_reset: initial state of every env at step index 0, first observation, zero reward / done
template <int G>
__global__ void reset_kernel(const __grid_constant__ DevParams P, const DevBuffers B) {
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const unsigned e_raw = tid / G;
    const int j = tid % G;
    const bool env_ok = e_raw < (unsigned)P.N;
    const unsigned e = env_ok ? e_raw : (unsigned)P.N - 1;
    const bool active = env_ok && j < P.M;
    const int jj = j < P.M ? j : P.M - 1;
    const size_t drone = (size_t)e * P.M + jj;
    DroneRegs d; float4 tg;
    reset_drone(P, e, (uint32_t)jj, 0u, d, tg);
    float adj[G];
#pragma unroll
    for (int kk = 0; kk < G; ++kk) adj[kk] = 0.0f;
    const bool with_adj = (P.feat & F_ADJ) != 0;
    if (with_adj) adjacency<G>(P, d.p, lane, j, adj);
    if (!active) return;
    store_state(B, drone, d);
    B.P4[drone] = make_float4(0, 0, 0, 0); B.P5[drone] = d.sp; B.P6[drone] = tg;
    write_obs<G>(P, B.obs, drone, d, v3(0, 0, 0), adj, with_adj);
    if (j == 0) { B.E0[e] = make_float4(0, 0, 0, __uint_as_float(0u)); B.gstep[e] = 0u; B.reward[e] = 0.0f; B.done[e] = 0; }
}

// recompute obs from the stored state (after mdg_set_state)
template <int G>
__global__ void refresh_obs_kernel(const __grid_constant__ DevParams P, const DevBuffers B) {
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const unsigned e_raw = tid / G;
    const int j = tid % G;
    const bool env_ok = e_raw < (unsigned)P.N;
    const unsigned e = env_ok ? e_raw : (unsigned)P.N - 1;
    const bool active = env_ok && j < P.M;
    const int jj = j < P.M ? j : P.M - 1;
    const size_t drone = (size_t)e * P.M + jj;
    DroneRegs d;
    load_state(B, drone, d);
    float adj[G];
#pragma unroll
    for (int kk = 0; kk < G; ++kk) adj[kk] = 0.0f;
    const bool with_adj = (P.feat & F_ADJ) != 0;
    if (with_adj) adjacency<G>(P, d.p, lane, j, adj);
    if (!active) return;
    write_obs<G>(P, B.obs, drone, d, euler_zyx(d.q), adj, with_adj);
}

// harness actions (stream 3): base * fma(hi - lo, u, lo), each operation rounded to fp32
__global__ void gen_actions_kernel(size_t n_drones_total, int M, uint32_t env_base, uint32_t seed_lo, uint32_t seed_hi, uint32_t t,
                                   float base, float lo, float hi, float4* __restrict__ out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_drones_total) return;
    const uint32_t e = (uint32_t)(i / M) + env_base, jd = (uint32_t)(i % M);
    const uint4 r = philox4x32_10(e, jd, t, STREAM_ACTION, seed_lo, seed_hi);
    const float span = __fsub_rn(hi, lo);
    out[i] = make_float4(__fmul_rn(base, __fmaf_rn(span, u01(r.x), lo)), __fmul_rn(base, __fmaf_rn(span, u01(r.y), lo)),
                         __fmul_rn(base, __fmaf_rn(span, u01(r.z), lo)), __fmul_rn(base, __fmaf_rn(span, u01(r.w), lo)));
}

}  // namespace mdg

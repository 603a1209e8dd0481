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
// sin/cos for |omega| h > 0.28 rad; the hot path uses the branch-free series (stage_torque, exp_half).
template <bool EXACT, bool EULER, int DEG>
__device__ __forceinline__ void integrate_rot(const DevParams& P, Q4& q, V3& w, V3 tau_b, V3 k1_tau, bool axisym) {
    auto ex = [](V3 phi) { return EXACT ? exp_half_exact(phi) : exp_half(phi); };
    if (!EULER) {
        const V3 w0 = w;
        const V3 k1 = v3(fmaf(-P.gyro[0], w0.y * w0.z, k1_tau.x), fmaf(-P.gyro[1], w0.z * w0.x, k1_tau.y),
                         axisym ? k1_tau.z : fmaf(-P.gyro[2], w0.x * w0.y, k1_tau.z));
        const V3 w2 = v3(fmaf(P.half_h, k1.x, w0.x), fmaf(P.half_h, k1.y, w0.y), fmaf(P.half_h, k1.z, w0.z));
        auto stage_half = [&](V3 ws) { return EXACT ? rot_inv(exp_half_exact(v3(P.half_h * ws.x, P.half_h * ws.y, P.half_h * ws.z)), tau_b)
                                                    : stage_torque<DEG>(P.rotA_half, P.rotB_half, ws, tau_b); };
        auto stage_full = [&](V3 ws) { return EXACT ? rot_inv(exp_half_exact(v3(P.h * ws.x, P.h * ws.y, P.h * ws.z)), tau_b)
                                                    : stage_torque<DEG>(P.rotA_full, P.rotB_full, ws, tau_b); };
        const V3 k2 = ang_acc(P, stage_half(w0), w2, axisym);
        const V3 w3 = v3(fmaf(P.half_h, k2.x, w0.x), fmaf(P.half_h, k2.y, w0.y), fmaf(P.half_h, k2.z, w0.z));
        const V3 k3 = ang_acc(P, stage_half(w2), w3, axisym);
        const V3 w4 = v3(fmaf(P.h, k3.x, w0.x), fmaf(P.h, k3.y, w0.y), fmaf(P.h, k3.z, w0.z));
        const V3 k4 = ang_acc(P, stage_full(w3), w4, axisym);
        const V3 ws = v3(w0.x + 2.0f * (w2.x + w3.x) + w4.x, w0.y + 2.0f * (w2.y + w3.y) + w4.y, w0.z + 2.0f * (w2.z + w3.z) + w4.z);
        q = qmul(q, EXACT ? exp_half_exact(v3(P.h_sixth * ws.x, P.h_sixth * ws.y, P.h_sixth * ws.z)) : exp_half_scaled<DEG>(P.expC, P.expS, ws));
        w = v3(fmaf(P.h_sixth, k1.x + 2.0f * (k2.x + k3.x) + k4.x, w0.x), fmaf(P.h_sixth, k1.y + 2.0f * (k2.y + k3.y) + k4.y, w0.y),
               fmaf(P.h_sixth, k1.z + 2.0f * (k2.z + k3.z) + k4.z, w0.z));
    } else {
        const V3 k1 = ang_acc(P, tau_b, w, axisym);
        w = v3(fmaf(P.h, k1.x, w.x), fmaf(P.h, k1.y, w.y), fmaf(P.h, k1.z, w.z));
        q = qmul(q, ex(v3(P.h * w.x, P.h * w.y, P.h * w.z)));
    }
    const float rn = rsqrt_fast(fmaf(q.w, q.w, fmaf(q.x, q.x, fmaf(q.y, q.y, q.z * q.z))));
    q.w *= rn; q.x *= rn; q.y *= rn; q.z *= rn;
}
// out-of-line copy for fast spins (|omega| h > 0.28 rad, i.e. > 67 rad/s at 240 Hz): rare, keeps the hot loop free of library calls
struct RotState { Q4 q; V3 w; };
template <bool EULER>
__device__ __noinline__ RotState integrate_rot_exact(const DevParams& P, Q4 q, V3 w, V3 tau_b, V3 k1_tau) {
    integrate_rot<true, EULER, 3>(P, q, w, tau_b, k1_tau, false);
    RotState r; r.q = q; r.w = w;
    return r;
}

// Shared-memory landing zone of one warp for one work item (32 lanes = 32 / G envs): every lane owns one
// 16-byte slot per plane, fills it with cp.async and is the only one to read it back, so no barrier of any
// kind is needed and the warps of a block never wait for each other.
struct WarpStage {
    float4 plane[9][32];           // P0..P6, the actions, E0 (the env word, one copy per lane)
    uint32_t gstep[32];
};
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Start the asynchronous copies of this lane's slots of lane-group row `wt` (32 / G envs; global -> shared, no registers held).
// dep: a zero the hardware cannot know to be zero, derived from the registers last read from S: the copies may overwrite S
// only once those reads have returned - a register dependency the address generation must wait for.
template <int G>
__device__ __forceinline__ void prefetch_item(const DevParams& P, const DevBuffers& B, const float4* actions, WarpStage& S,
                                              unsigned wt, int lane, int jj, int act, unsigned dep) {
    const unsigned e_raw = wt * (32u / G) + (unsigned)lane / G;
    const unsigned e = (e_raw < (unsigned)P.N ? e_raw : (unsigned)P.N - 1) + dep;
    const size_t drone = (size_t)e * P.M + jj;
    cp_async16(&S.plane[0][lane], B.P0 + drone);
    cp_async16(&S.plane[1][lane], B.P1 + drone);
    cp_async16(&S.plane[2][lane], B.P2 + drone);
    cp_async16(&S.plane[3][lane], B.P3 + drone);
    if (act == 1 || act == 2 || act == 5) cp_async16(&S.plane[4][lane], B.P4 + drone);   // actions with an attitude loop
    if (act == 1) cp_async16(&S.plane[5][lane], B.P5 + drone);
    cp_async16(&S.plane[6][lane], B.P6 + drone);
    cp_async16(&S.plane[7][lane], actions + drone);
    cp_async16(&S.plane[8][lane], B.E0 + e);
    cp_async4(&S.gstep[lane], B.gstep + e);
}


// ---- lane-generic rotation update and substep ---------------------------------------------------------------------------
template <int N> struct NPTag {};
template <int NP> struct Lanes;
template <> struct Lanes<1> { typedef float T; };
template <> struct Lanes<2> { typedef F2 T; };
__device__ __forceinline__ float pack_lanes(NPTag<1>, float a, float) { return a; }
__device__ __forceinline__ F2 pack_lanes(NPTag<2>, float a, float b) { return pk(a, b); }
__device__ __forceinline__ float half_of(float x, int) { return x; }
__device__ __forceinline__ float half_of(F2 x, int h) { return h ? hi_(x) : lo_(x); }
__device__ __forceinline__ bool half_of(bool m, int) { return m; }
__device__ __forceinline__ bool half_of(B2 m, int h) { return h ? m.hi : m.lo; }
__device__ __forceinline__ bool any_(bool m) { return m; }
__device__ __forceinline__ bool any_(B2 m) { return m.lo || m.hi; }
template <class T> __device__ __forceinline__ V3T<float> half3(V3T<T> a, int h) { return v3t<float>(half_of(a.x, h), half_of(a.y, h), half_of(a.z, h)); }

// angular acceleration J^-1 (tau_body - w x J w); axisym: J_xx == J_yy, the z component has no gyroscopic term
template <class T> __device__ __forceinline__ V3T<T> ang_acc_t(const DevParams& P, V3T<T> tb, V3T<T> w, bool axisym) {
    return v3t<T>(fma_(P.invJ[0], tb.x, mul_(P.ngyro[0], mul_(w.y, w.z))),
                  fma_(P.invJ[1], tb.y, mul_(P.ngyro[1], mul_(w.z, w.x))),
                  axisym ? fma_(P.invJ[2], tb.z, 0.0f) : fma_(P.invJ[2], tb.z, mul_(P.ngyro[2], mul_(w.x, w.y))));   // an fma with a zero addend, not
    // a multiply: the product is summed with the other stages' right away, and ptxas contracts a PACKED multiply-add pair into one
    // FFMA2 (it never does so for the scalar mul.rn / add.rn), which would make the two instantiations round differently
}
// S8 rotation, series form (the hot path): classical RK4 on (q, w_body) with the torque frozen in the world frame (MJC* modes)
// or explicit Euler (DYN).  The stage orientation is q0 (x) dq, so the body-frame torque at a stage is R(dq)^T tau_b and q0
// itself is only needed for the final update.  Valid for |omega| h below P.w2_exact; the caller re-does faster spins exactly.
template <bool EULER, int DEG, class T>
__device__ __forceinline__ void integrate_rot_t(const DevParams& P, Q4T<T>& q, V3T<T>& w, V3T<T> tau_b, V3T<T> k1_tau, bool axisym) {
    if (!EULER) {
        const V3T<T> w0 = w;
        const V3T<T> k1 = v3t<T>(fma_(P.ngyro[0], mul_(w0.y, w0.z), k1_tau.x), fma_(P.ngyro[1], mul_(w0.z, w0.x), k1_tau.y),
                                 axisym ? k1_tau.z : fma_(P.ngyro[2], mul_(w0.x, w0.y), k1_tau.z));
        const V3T<T> w2 = v3t<T>(fma_(P.half_h, k1.x, w0.x), fma_(P.half_h, k1.y, w0.y), fma_(P.half_h, k1.z, w0.z));
        const V3T<T> k2 = ang_acc_t(P, stage_torque_t<DEG>(P.rotnA_half, P.rotB_half, w0, tau_b), w2, axisym);
        const V3T<T> w3 = v3t<T>(fma_(P.half_h, k2.x, w0.x), fma_(P.half_h, k2.y, w0.y), fma_(P.half_h, k2.z, w0.z));
        const V3T<T> k3 = ang_acc_t(P, stage_torque_t<DEG>(P.rotnA_half, P.rotB_half, w2, tau_b), w3, axisym);
        const V3T<T> w4 = v3t<T>(fma_(P.h, k3.x, w0.x), fma_(P.h, k3.y, w0.y), fma_(P.h, k3.z, w0.z));
        const V3T<T> k4 = ang_acc_t(P, stage_torque_t<DEG>(P.rotnA_full, P.rotB_full, w3, tau_b), w4, axisym);
        // Eq.7 with the RK4 mean of the stage rates, (w0 + 2 w2 + 2 w3 + w4) / 6 = w0 + h/6 (k1 + k2 + k3), and the rate update
        // w0 + h/6 (k1 + 2 k2 + 2 k3 + k4) share k2 + k3 and k1 + k2 + k3
        const V3T<T> k23 = v3t<T>(add_(k2.x, k3.x), add_(k2.y, k3.y), add_(k2.z, k3.z));
        const V3T<T> ks = v3t<T>(add_(k1.x, k23.x), add_(k1.y, k23.y), add_(k1.z, k23.z));
        const V3T<T> wm = v3t<T>(fma_(P.h_sixth, ks.x, w0.x), fma_(P.h_sixth, ks.y, w0.y), fma_(P.h_sixth, ks.z, w0.z));
        q = qmul_t(q, exp_half_scaled_t<DEG>(P.expCm, P.expSm, wm));
        w = v3t<T>(fma_(P.h_sixth, add_(add_(ks.x, k23.x), k4.x), w0.x), fma_(P.h_sixth, add_(add_(ks.y, k23.y), k4.y), w0.y),
                   fma_(P.h_sixth, add_(add_(ks.z, k23.z), k4.z), w0.z));
    } else {
        const V3T<T> k1 = ang_acc_t(P, tau_b, w, axisym);
        w = v3t<T>(fma_(P.h, k1.x, w.x), fma_(P.h, k1.y, w.y), fma_(P.h, k1.z, w.z));
        q = qmul_t(q, exp_half_t(v3t<T>(mul_(P.h, w.x), mul_(P.h, w.y), mul_(P.h, w.z))));
    }
    const T rn = rsqrt_(fma_(q.w, q.w, fma_(q.x, q.x, fma_(q.y, q.y, mul_(q.z, q.z)))));   // (1.5 - 0.5 |q|^2 instead of the MUFU: measured slower, the FP32 pipe is the busy one)
    q.w = mul_(q.w, rn); q.x = mul_(q.x, rn); q.y = mul_(q.y, rn); q.z = mul_(q.z, rn);
}
// fast spins (|omega| h above the series' range): redo the rotation update from the start-of-substep values with the library
// sin / cos, out of line, one lane (half) at a time; never taken by the benchmark workloads
template <bool EULER> __device__ __forceinline__ void redo_fast_spin(const DevParams& P, bool fast, Q4T<float>& q, V3T<float>& w, Q4T<float> q0, V3T<float> w0,
                                                                      V3T<float> tau_b, V3T<float> k1_tau) {
    if (fast) {
        Q4 a; a.w = q0.w; a.x = q0.x; a.y = q0.y; a.z = q0.z;
        const RotState rs = integrate_rot_exact<EULER>(P, a, v3(w0.x, w0.y, w0.z), v3(tau_b.x, tau_b.y, tau_b.z), v3(k1_tau.x, k1_tau.y, k1_tau.z));
        q.w = rs.q.w; q.x = rs.q.x; q.y = rs.q.y; q.z = rs.q.z; w.x = rs.w.x; w.y = rs.w.y; w.z = rs.w.z;
    }
}
template <bool EULER> __device__ __forceinline__ void redo_fast_spin(const DevParams& P, B2 fast, Q4T<F2>& q, V3T<F2>& w, Q4T<F2> q0, V3T<F2> w0,
                                                                      V3T<F2> tau_b, V3T<F2> k1_tau) {
    if (fast.lo || fast.hi) {
        float r[2][7];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            Q4T<float> qh; qh.w = half_of(q.w, h); qh.x = half_of(q.x, h); qh.y = half_of(q.y, h); qh.z = half_of(q.z, h);
            V3T<float> wh = v3t<float>(half_of(w.x, h), half_of(w.y, h), half_of(w.z, h));
            Q4T<float> q0h; q0h.w = half_of(q0.w, h); q0h.x = half_of(q0.x, h); q0h.y = half_of(q0.y, h); q0h.z = half_of(q0.z, h);
            redo_fast_spin<EULER>(P, h ? fast.hi : fast.lo, qh, wh, q0h, v3t<float>(half_of(w0.x, h), half_of(w0.y, h), half_of(w0.z, h)),
                                  v3t<float>(half_of(tau_b.x, h), half_of(tau_b.y, h), half_of(tau_b.z, h)),
                                  v3t<float>(half_of(k1_tau.x, h), half_of(k1_tau.y, h), half_of(k1_tau.z, h)));
            r[h][0] = qh.w; r[h][1] = qh.x; r[h][2] = qh.y; r[h][3] = qh.z; r[h][4] = wh.x; r[h][5] = wh.y; r[h][6] = wh.z;
        }
        q.w = pk(r[0][0], r[1][0]); q.x = pk(r[0][1], r[1][1]); q.y = pk(r[0][2], r[1][2]); q.z = pk(r[0][3], r[1][3]);
        w.x = pk(r[0][4], r[1][4]); w.y = pk(r[0][5], r[1][5]); w.z = pk(r[0][6], r[1][6]);
    }
}

// What a lane integrates over the substeps: one drone (T = float) or the same drone index of two envs (T = F2).
template <class T> struct Body {
    V3T<T> p; Q4T<T> q; V3T<T> v, w;                              // state, w in the body frame
    V3T<T> tau_b, k1_tau, a0;                                     // frozen over a substep: Eq.1-3 torque, J^-1 tau; wind force / m - g z
    T thrust, cxy, dcz, gndT, ndwc;                               // thrust, Eq.5 / Eq.4 coefficients x rotor terms, -Eq.6 coefficient: all / m
};
// One physics substep (S4-S8): world-frame force from the start-of-substep state, then the free-body update with the wrench
// frozen.  Returns "went through the floor" (clamped).  The downwash exchange is a shuffle inside the G-lane group.
template <class T> struct SubstepFlags { typename LaneOps<T>::mask below, fast; };   // went through the floor (clamped); spun too fast for the series
__device__ __forceinline__ bool inline_redo(float) { return true; }
__device__ __forceinline__ bool inline_redo(F2) { return false; }
template <int G, int FEAT, int DEG, class T>
__device__ __forceinline__ SubstepFlags<T> substep(const DevParams& P, Body<T>& s, int j, bool full_group) {
    using F = Feat<FEAT>;
    // b = R(q) z: thrust is T b, and Eq.5's R diag(c_xy, c_xy, c_z) R^T v = c_xy v + (c_z - c_xy)(b.v) b
    const T bx = mul_(2.0f, fma_(s.q.x, s.q.z, mul_(s.q.w, s.q.y)));
    const T by = mul_(2.0f, fma_(s.q.y, s.q.z, mul_(neg_(s.q.w), s.q.x)));
    const T bz = fma_(-2.0f, fma_(s.q.x, s.q.x, mul_(s.q.y, s.q.y)), 1.0f);
    // every coefficient already carries 1 / m and a0 = F_wind / m - g z, so the sums below are the acceleration itself
    V3T<T> Fw;
    if (F::has(P, F_DRAG)) {
        const T sc = fma_(s.dcz, fma_(bx, s.v.x, fma_(by, s.v.y, mul_(bz, s.v.z))), s.thrust);
        Fw = v3t<T>(fma_(sc, bx, fma_(s.cxy, s.v.x, s.a0.x)), fma_(sc, by, fma_(s.cxy, s.v.y, s.a0.y)), fma_(sc, bz, fma_(s.cxy, s.v.z, s.a0.z)));
    } else Fw = v3t<T>(fma_(s.thrust, bx, s.a0.x), fma_(s.thrust, by, s.a0.y), fma_(s.thrust, bz, s.a0.z));
    if (F::has(P, F_GND)) {                                       // Eq.4, gated on body z pointing up
        const T hgt = max_(s.p.z, P.h_clip);
        const T gain = mul_(s.gndT, rcp_(mul_(hgt, hgt)));
        Fw.z = add_(Fw.z, sel_(gt_(bz, 0.0f), gain, 0.0f));
    }
    if (G > 1 && F::has(P, F_DW)) {                               // Eq.6 over every drone above this one
        // With b' = sqrt(2 ln 2) beta: exp(-dxy^2 / 2 beta^2) = 2^(-dxy^2 / b'^2) and alpha = C1 (r_p/4)^2 / dz_e^2: two MUFU
        // reciprocals (the XU pipe is idle most of the time; one shared reciprocal costs three more multiplies on the FP32 pipe).
        // The ramp saturate(dz / dz_clip) is 0 for dz <= 0, which also gates "k above this drone";
        // b'^2 is floored (beta^2 >= 1e-12), which reproduces the beta -> 0 rule of DESIGN.md Q9.
        // Pairs are shared out: in round r < G/2 lane j evaluates the pair (j, j + r mod G) once for both ends -
        // the force goes to whichever drone is lower, the partner's share travels back by one shuffle - and in
        // round G/2 both ends evaluate their common pair and each keeps its own share.
        T dw = LaneOps<T>::bc(0.0f);
#pragma unroll
        for (int r = 1; r <= G / 2; ++r) {
            const int src = j + r;                                 // logical lane inside the G-wide segment (taken mod G)
            const T ox = shfl_(s.p.x, src, G), oy = shfl_(s.p.y, src, G), oz = shfl_(s.p.z, src, G);
            const T dz = sub_(oz, s.p.z), dx = sub_(ox, s.p.x), dy = sub_(oy, s.p.y);
            const T dxy2 = fma_(dx, dx, mul_(dy, dy));
            const T adz = abs_(dz);
            const T dze = max_(adz, P.dz_floor);
            const T ramp = sat_(mul_(adz, P.inv_dz_clip));
            const T bs = fma_(P.dw_C2s, dze, P.dw_C3s);
            const T b2 = max_(mul_(bs, bs), P.dw_b2_min), z2 = mul_(dze, dze);
            const T ex = ex2n_(mul_(dxy2, rcp_(b2)));
            const T al = mul_(ramp, rcp_(z2));
            const bool on = full_group || (j < P.M && ((j + r) & (G - 1)) < P.M);
            const T f = sel_(and_(lt_(dxy2, 100.0f), on), mul_(al, ex), 0.0f);
            const typename LaneOps<T>::mask above = gt_(dz, 0.0f);   // the partner is above this drone
            if (r < G / 2) {
                const T back = shfl_(sel_(above, 0.0f, f), j + G - r, G);
                dw = add_(dw, add_(sel_(above, f, 0.0f), back));
            } else dw = add_(dw, sel_(above, f, 0.0f));
        }
        Fw.z = fma_(s.ndwc, dw, Fw.z);
    }
    const V3T<T> acc = Fw;

    // S8 integrate with the wrench frozen in the world frame
    const typename LaneOps<T>::mask fast_spin = gt_(dot3(s.w, s.w), P.w2_exact[DEG - 2]);
    const Q4T<T> q0 = s.q;
    const V3T<T> w0 = s.w;
    if (!F::has(P, F_EULER)) {
        s.p.x = fma_(P.half_h2, acc.x, fma_(P.h, s.v.x, s.p.x));
        s.p.y = fma_(P.half_h2, acc.y, fma_(P.h, s.v.y, s.p.y));
        s.p.z = fma_(P.half_h2, acc.z, fma_(P.h, s.v.z, s.p.z));
        s.v.x = fma_(P.h, acc.x, s.v.x); s.v.y = fma_(P.h, acc.y, s.v.y); s.v.z = fma_(P.h, acc.z, s.v.z);
        integrate_rot_t<false, DEG>(P, s.q, s.w, s.tau_b, s.k1_tau, F::has(P, F_AXISYM));
        if (inline_redo(s.p.x)) redo_fast_spin<false>(P, fast_spin, s.q, s.w, q0, w0, s.tau_b, s.k1_tau);
    } else {                                                       // DYN: explicit Euler
        s.v.x = fma_(P.h, acc.x, s.v.x); s.v.y = fma_(P.h, acc.y, s.v.y); s.v.z = fma_(P.h, acc.z, s.v.z);
        s.p.x = fma_(P.h, s.v.x, s.p.x); s.p.y = fma_(P.h, s.v.y, s.p.y); s.p.z = fma_(P.h, s.v.z, s.p.z);
        integrate_rot_t<true, DEG>(P, s.q, s.w, s.tau_b, s.k1_tau, F::has(P, F_AXISYM));
        if (inline_redo(s.p.x)) redo_fast_spin<true>(P, fast_spin, s.q, s.w, q0, w0, s.tau_b, s.k1_tau);
    }
    const typename LaneOps<T>::mask below = lt_(s.p.z, 0.0f);       // floor
    s.v.z = sel_(below, max_(s.v.z, 0.0f), s.v.z);
    s.p.z = sel_(below, 0.0f, s.p.z);
    SubstepFlags<T> fl; fl.below = below; fl.fast = fast_spin;
    return fl;
}
// Two envs per lane keep the hot loop free of the exact path: a warp in which any lane spun too fast during the step redoes the
// step's K substeps one env slot at a time with the one-drone code (same arithmetic: the result is what one env per lane
// computes), from the start-of-step state, which is still what global memory holds.  Out of line, never taken by the benchmarks.
struct RedoOut { float s[13]; bool hit; };
template <int G, int FEAT, int DEG>
__device__ __noinline__ RedoOut redo_item_exact(const DevParams& P, const float4* p0, const float4* p1, const float4* p2, const float4* p3, Body<float> b,
                                                int j, bool full_group) {
    const float4 a0 = *p0, a1 = *p1, a2 = *p2, a3 = *p3;          // the step's stores have not happened yet
    b.p = v3t<float>(a0.x, a0.y, a0.z); b.q.w = a0.w; b.q.x = a1.x; b.q.y = a1.y; b.q.z = a1.z;
    b.v = v3t<float>(a1.w, a2.x, a2.y); b.w = v3t<float>(a2.z, a2.w, a3.x);
    RedoOut o; o.hit = false;
    for (int k = 0; k < P.K; ++k) o.hit |= substep<G, FEAT, DEG>(P, b, j, full_group).below;
    o.s[0] = b.p.x; o.s[1] = b.p.y; o.s[2] = b.p.z; o.s[3] = b.q.w; o.s[4] = b.q.x; o.s[5] = b.q.y; o.s[6] = b.q.z;
    o.s[7] = b.v.x; o.s[8] = b.v.y; o.s[9] = b.v.z; o.s[10] = b.w.x; o.s[11] = b.w.y; o.s[12] = b.w.z;
    return o;
}

// S7: one AR(1) step of an env's gust, w <- alpha w + sigma sqrt(1 - alpha^2) xi, xi from one Philox draw at
// (env, ~0, t, stream 2).  Box-Muller on (1 - u_a, u_b): r = sqrt(-2 ln(1 - u_a)) = sqrt(-2 ln2 lg2(1 - u_a)); 1 - u_a is exact
// in fp32; cos / sin(2 pi u_b) = -cos / sin(2 pi (u_b - 1/2)) keeps the MUFU argument in [-pi, pi).
__device__ __forceinline__ V3 gust_update(const DevParams& P, unsigned e, uint32_t t, V3 w, float wa, float wg) {
    const uint4 r = philox4x32_10(e + P.env_base, 0xFFFFFFFFu, t, STREAM_WIND, P.seed_lo, P.seed_hi);
    const float r1 = -fast_sqrt(__fmul_rn(-1.38629436f, lg2_fast(__fsub_rn(1.0f, u01(r.x))))), r2 = -fast_sqrt(__fmul_rn(-1.38629436f, lg2_fast(__fsub_rn(1.0f, u01(r.z)))));
    const float a1 = __fmul_rn(6.28318531f, __fsub_rn(u01(r.y), 0.5f)), a2 = __fmul_rn(6.28318531f, __fsub_rn(u01(r.w), 0.5f));
    return v3(fmaf(wa, w.x, __fmul_rn(wg, __fmul_rn(r1, cos_fast(a1)))), fmaf(wa, w.y, __fmul_rn(wg, __fmul_rn(r1, sin_fast(a1)))),
              fmaf(wa, w.z, __fmul_rn(wg, __fmul_rn(r2, cos_fast(a2)))));
}

// What one lane carries for one of its NP env slots from the prologue to the epilogue of a work item.
struct Slot {
    unsigned e; bool active; size_t drone;
    DroneRegs d; float4 tg, act4, env4; uint32_t t;
    float4 dr0, dr1, dr2, dr3;                                    // this episode's DR factors (read-mostly, plain loads)
    V3 Fwind; float4 gust_out;                                    // wind force held over the substeps; E1 after this step (MDG_WIND_GUST)
    float n[4], n_later[4], n_act[4], lag_gain; int sw, d_obs;    // rotor commands (now / after the latency switch), rotor speeds under lag
    float kf_e, kappa_e, inv_sJ, inv_m_e, g_e, dwc_e, nmax;       // the true vehicle of this episode (Table 4)
    DecodeMid mid;                                                // controller actions: what decode_front leaves for control_loops
    bool hit; Sensed snap;
};

// One control step of every env.  Persistent warps: each loops over work items of
// NP * 32 / G envs; lane -> (lane-in-group j, NP envs: slot h holds env (item * NP + h) * 32 / G + lane / G).  With NP = 2 the
// substeps of a lane's two drones run as packed FP32 pairs (mdg_dev.cuh: F2), everything else once per slot.  While an item is
// integrated, the next item's state planes, actions and per-env words are already on their way into shared memory (cp.async
// into the warp's landing zone), so HBM latency and bandwidth overlap the arithmetic instead of alternating with it.
// MINB = resident blocks of 128 threads per SM the register allocation must allow.
template <int G, int FEAT, int MINB, int NP>
__global__ void __launch_bounds__(128, MINB) step_kernel(const __grid_constant__ DevParams P, const DevBuffers B,
                                                         const float4* __restrict__ actions) {
    using F = Feat<FEAT>;
    using T = typename Lanes<NP>::T;
    static_assert(NP == 1 || FEAT >= 0, "two envs per lane need a compile-time feature word");
    static_assert(NP == 1 || !(FEAT & (F_MLAG | F_LAT)), "motor lag and the latency rows switch rotor commands inside the substep loop: one env per lane");
    // series degree of the rotation update: 2 where the specialisation's controller keeps the body rates small (PID / VEL)
    constexpr int DEG = (FEAT >= 0 && (((FEAT >> F_ACT_SHIFT) & 7) == 1 || ((FEAT >> F_ACT_SHIFT) & 7) == 2)) ? 2 : 3;
    extern __shared__ __align__(16) unsigned char smem_raw[];     // [warps per block][NP] WarpStage, then the stash (host sizes it)
    WarpStage* const S = reinterpret_cast<WarpStage*>(smem_raw);
    // Behind the landing zones: the warp's stash, one 16-byte slot per lane, env slot and parked quantity.  What only the epilogue
    // needs (controller memory, target, env word, ...) waits there during the substeps, so the loop holds nothing but the
    // integrated state and the frozen wrench in registers, and the landing zone is free for the next item right away.
    const int obs_kin20 = F::obs(P) == 2;
    const int act1 = F::act(P) == 1;
    const int pid_i = (F::act(P) == 1 || F::act(P) == 2 || F::act(P) == 5) ? 1 : 0;
    const int iIP = 0, iTG = 1, iENV = 2, iIE = 3, iSP = 3 + pid_i, iACT = 3 + pid_i + act1;
    const int n_stash = 3 + pid_i + act1 + obs_kin20;             // the host sizes the shared memory with the same count
    float4* const stash0 = reinterpret_cast<float4*>(smem_raw + (size_t)(blockDim.x >> 5) * NP * sizeof(WarpStage));
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const unsigned wpb = blockDim.x >> 5;
    const unsigned tw = gridDim.x * wpb;                          // persistent warps of this launch
    const unsigned epi = NP * (32u / G);                          // envs per work item
    const unsigned n_items = ((unsigned)P.N + epi - 1) / epi;
    const int j = lane % G;
    const bool full_group = F::has(P, F_FULL);
    const int jj = (full_group || j < P.M) ? j : P.M - 1;
    const bool pid = F::act(P) == 1 || F::act(P) == 2 || F::act(P) == 5;   // actions with an attitude loop (I_eta in P4)
    // Programmatic dependent launch.  P.chain == 0: wait here until the previous kernel of the stream has completed
    // and its writes are visible (nothing above touches memory).  P.chain == 1 (mdg_step_chained / the inner launches of
    // mdg_step_many: the previous operation on this handle was step number P.seq - 1, launched on the same stream or in the
    // same capture, and the caller guarantees that the actions were complete before that step was enqueued): no grid-wide
    // wait at all; the dependency is per work item instead - item i may start as soon as the previous step has published
    // item i (item_seq[i] == P.seq - 1, release/acquire), so the drain of one step overlaps the ramp-up of the next.
    // Deadlock-free: this grid only starts once every block of the previous grid is resident (or done), and nothing here
    // is waited on by that grid.  Sequence numbers are kernel parameters: in a replayed CUDA graph the first launch has
    // chain == 0 and publishes its (baked) number for every item, so the second finds what it expects in every replay.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t seq = P.seq;
    const bool chain = P.chain != 0;
    if (!chain) asm volatile("griddepcontrol.wait;" ::: "memory");
    // Every warp starts on the item of its own index (known without a memory round trip: the blocks of a launch start
    // within a microsecond of each other, whatever they wait for first is paid by all of them); the others are handed out
    // by an atomic ticket (item = tw + ticket; self-resetting: atomicInc wraps to 0 after the n_items grabs of one launch -
    // n_items - tw items and one miss per warp; four dispensers take turns so that chained launches never share one), so SMs
    // that run faster or host fewer long warps simply take more items.
    const unsigned wrap = n_items - 1u;
    unsigned* const dispenser = B.ticket + (seq & 3u);
    // Everything with a long latency on the per-item path is issued one item early and consumed late: the ticket
    // of item n+2 is drawn (lane 0, atomic) when item n starts and read after its substeps; the "previous step
    // has published this item" flag of item n+2 is then probed (ld.acquire) and only re-polled at the prefetch
    // of item n+2 if that probe came too early; an item's own flag is published (fence + st.release) just before
    // the NEXT item's stores, when its stores have long been acknowledged.
    const unsigned want = seq - 1u;
    auto draw = [&](bool go) { unsigned v = 0xFFFFFFFFu; if (lane == 0 && go) v = tw + atomicInc(dispenser, wrap); return v; };   // lane 0 holds it
    auto take = [&](unsigned drawn_l0) { return __shfl_sync(MDG_FULL, drawn_l0, 0); };
    auto probe = [&](unsigned item_l0) {                        // lane 0: one acquire load of the item's flag
        unsigned got = want;
        if (chain && lane == 0 && item_l0 < n_items) asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(got) : "l"(B.item_seq + item_l0) : "memory");
        return got;
    };
    auto await_item = [&](unsigned item, unsigned probed_l0) {  // the previous step has finished this item
        if (chain) {
            if (lane == 0 && probed_l0 != want) {
                unsigned got, spins = 0;
                for (;;) {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(got) : "l"(B.item_seq + item) : "memory");
                    if (got == want) break;
                    __nanosleep(64);
                    if (++spins > (1u << 24)) __trap();          // fail loudly instead of hanging
                }
            }
            __syncwarp();
        }
    };
    // publication of an item = fence over every lane's stores (issued before the substeps of the next item, whose
    // arithmetic hides the fence's round trip to L2) + a relaxed store of the sequence number (after them)
    auto publish_flag = [&](unsigned item) {
        __syncwarp();
        if (lane == 0) asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(B.item_seq + item), "r"(seq) : "memory");
    };
    // Grids that do not fill the device hold one warp per item: no ticket is drawn at all, so any number of such launches
    // may be in flight at once (each item still waits for its predecessor's flag).
    const bool static_items = P.static_items != 0;
    unsigned wt = blockIdx.x * wpb + wib;
    if (wt >= n_items) return;                                    // only in grids that do not fill the device (static_items)
    // start-up: the first item's flag probe and the first ticket are in flight together, the item's copies start as soon as
    // the flag is in (every warp of a launch pays this once, a good part of its life when a launch gives it two or three items)
    const unsigned probed_first = probe(wt);
    const unsigned drawn_first = draw(!static_items);
    await_item(wt, probed_first);
    auto prefetch = [&](unsigned item, unsigned dep) {
#pragma unroll
        for (int h = 0; h < NP; ++h) prefetch_item<G>(P, B, actions, S[wib * NP + h], item * NP + h, lane, jj, F::act(P), dep);
        cp_async_commit();
    };
    prefetch(wt, 0u);
    unsigned wt_next = static_items ? 0xFFFFFFFFu : take(drawn_first);   // a warp stops drawing after its first miss
    unsigned probed_next = probe(wt_next);
    // Items whose flags are still to be published.  One fence covers two items: the consumer (the next step) reaches
    // an item a whole step later, so publishing it one item late costs nothing and halves the fences.
    unsigned pending = 0xFFFFFFFFu, pending2 = 0xFFFFFFFFu;
#pragma unroll 1
    for (;;) {
    const unsigned drawn_l0 = draw(wt_next < n_items);            // ticket of the item after next, in flight
    Slot sl[NP];
    unsigned touched = 0u;                                        // OR of one word of every shared-memory read of this item
    cp_async_wait_all();
#pragma unroll
    for (int h = 0; h < NP; ++h) {
        Slot& s = sl[h];
        const unsigned e_raw = (wt * NP + h) * (32u / G) + (unsigned)lane / G;
        const bool env_ok = e_raw < (unsigned)P.N;
        s.e = env_ok ? e_raw : (unsigned)P.N - 1;                 // idle lanes shadow the last env (no stores)
        s.active = env_ok && (full_group || j < P.M);
        s.drone = (size_t)s.e * P.M + jj;
        const WarpStage& W = S[wib * NP + h];
        const float4 a = W.plane[0][lane], b = W.plane[1][lane], c = W.plane[2][lane], f = W.plane[3][lane];
        s.d.p = v3(a.x, a.y, a.z); s.d.q.w = a.w; s.d.q.x = b.x; s.d.q.y = b.y; s.d.q.z = b.z;
        s.d.v = v3(b.w, c.x, c.y); s.d.w = v3(c.z, c.w, f.x); s.d.Ip = v3(f.y, f.z, f.w);
        if (pid) {
            const float4 i4 = W.plane[4][lane];
            s.d.Ie = v3(i4.x, i4.y, i4.z);
            if (F::act(P) == 1) s.d.sp = W.plane[5][lane];
        }
        s.tg = W.plane[6][lane];
        s.act4 = W.plane[7][lane];
        s.env4 = W.plane[8][lane];
        s.t = W.gstep[lane] + 1u;
        touched |= __float_as_uint(a.x) | __float_as_uint(b.x) | __float_as_uint(c.x) | __float_as_uint(f.x) | __float_as_uint(s.tg.x) |
                   __float_as_uint(s.act4.x) | __float_as_uint(s.env4.x) | s.t;
        if (pid) touched |= __float_as_uint(s.d.Ie.x) | (F::act(P) == 1 ? __float_as_uint(s.d.sp.x) : 0u);
        s.dr0 = make_float4(1, 1, 1, 1); s.dr1 = s.dr0; s.dr2 = s.dr0; s.dr3 = s.dr0;
        if (F::has(P, F_DR)) { s.dr0 = B.R0[s.drone]; s.dr1 = B.R1[s.drone]; s.dr2 = B.R2[s.drone]; s.dr3 = B.R3[s.drone]; }
    }
    // the next item starts coming now, into the same landing zone: its contents are all in registers (`touched` makes the copies'
    // addresses depend on them, so no copy can overtake a read)
    if (wt_next < n_items) { await_item(wt_next, probed_next); prefetch(wt_next, touched & P.zero); }

    const bool dr = F::has(P, F_DR);
    const bool lag = F::has(P, F_MLAG);
    // Two envs per lane and at least two lanes per env: the AR(1) gust of an env is the same for all its lanes, so lane j draws
    // it for env slot j & 1 only and the group's lanes 0 and 1 hand their results round (six shuffles instead of a second
    // Philox + Box-Muller per lane; the arithmetic is gust_update either way).
    const bool share_gust = NP == 2 && G >= 2 && F::has(P, F_WIND) && !F::has(P, F_WIND_MIX);
    float gust_x[NP], gust_y[NP], gust_z[NP];
    if (share_gust) {
        const int hs = j & 1;
        const Slot& s0 = sl[0]; const Slot& s1 = sl[NP - 1];
        const V3 mine = gust_update(P, hs ? s1.e : s0.e, hs ? s1.t : s0.t,
                                    hs ? v3(s1.env4.x, s1.env4.y, s1.env4.z) : v3(s0.env4.x, s0.env4.y, s0.env4.z), P.wind_alpha, P.wind_gain);
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            gust_x[h] = __shfl_sync(MDG_FULL, mine.x, h, G); gust_y[h] = __shfl_sync(MDG_FULL, mine.y, h, G); gust_z[h] = __shfl_sync(MDG_FULL, mine.z, h, G);
        }
    }
#pragma unroll
    for (int h = 0; h < NP; ++h) {
        Slot& s = sl[h];
        DroneRegs& d = s.d;
        float4& env4 = s.env4;
        const unsigned e = s.e;
        const uint32_t t = s.t;
        const float4 act4 = s.act4;
        const size_t drone = s.drone;
        const bool active = s.active;
        // S7 wind gust: one AR(1) update per env and control step (gust_update), force held over the substeps.
        V3 Fwind = v3(0, 0, 0);
        float4 gust_out = make_float4(0, 0, 0, 1.0f);                  // E1 after this step (generic kernel, MDG_WIND_GUST only)
        if (F::has(P, F_WIND)) {
            // components (MDG_WIND_*): the benchmark configs run the AR(1) gust alone (wmask == 1 folds at compile time)
            const int wmask = F::has(P, F_WIND_MIX) ? P.wind_mask : 1;
            V3 u = v3(0, 0, 0);                                        // air velocity
            if (wmask & 1) {
                if (share_gust) { env4.x = gust_x[h]; env4.y = gust_y[h]; env4.z = gust_z[h]; }   // drawn once per env, above
                else {
                    float wa = P.wind_alpha, wg = P.wind_gain;
                    if (F::has(P, F_WIND_MIX) && P.dryden_x > 0.0f) {                  // PAPER.md:202 (Q50): L_u(h) at the env's mean altitude,
                        const float hm = fmaxf(group_sum<G>((full_group || j < P.M) ? d.p.z : 0.0f) * P.inv_M, P.dryden_h_min);   // alpha = exp(-dt V / L)
                        const float x = P.dryden_x * powf(fmaf(8.23e-4f, hm, 0.177f), 1.2f) / hm;
                        wa = expf(-x);
                        wg = P.wind_sigma * sqrtf(-expm1f(-2.0f * x));    // sigma sqrt(1 - alpha^2) without the cancellation
                    }
                    const V3 wn = gust_update(P, e, t, v3(env4.x, env4.y, env4.z), wa, wg);
                    env4.x = wn.x; env4.y = wn.y; env4.z = wn.z;
                }
                u = v3(env4.x, env4.y, env4.z);
            }
            if (wmask & 2) { u.x += P.wind_const[0]; u.y += P.wind_const[1]; u.z += P.wind_const[2]; }
            if (wmask & 4) {                                           // PAPER.md:201 impulses (Q42), state in E1
                float4 gs = B.E1[e];
                constexpr float GUST_END = 1.0f - 1e-4f;               // Q42: over at phase 1 - 1e-4, so that a duration of a whole number of steps is no rounding tie
                if (gs.w >= GUST_END) {                                // none running: trigger with probability gust_prob
                    const uint4 r = philox4x32_10(e + P.env_base, 0xFFFFFFFFu, t, STREAM_GUST, P.seed_lo, P.seed_hi);
                    if (u01(r.x) < P.gust_prob) {
                        const float amp = P.gust_max * u01(r.y), z = fmaf(2.0f, u01(r.z), -1.0f);
                        const float rxy = sqrtf(fmaxf(fmaf(-z, z, 1.0f), 0.0f));
                        float sp, cp;
                        sincospif(2.0f * u01(r.w), &sp, &cp);
                        gs = make_float4(amp * rxy * cp, amp * rxy * sp, amp * z, 0.0f);
                    }
                }
                if (gs.w < GUST_END) {                                 // envelope sin(pi s), s advances by dt_c / duration
                    const float es = sinpif(gs.w);
                    u.x = fmaf(gs.x, es, u.x); u.y = fmaf(gs.y, es, u.y); u.z = fmaf(gs.z, es, u.z);
                    gs.w += P.gust_ds;
                }
                gust_out = gs;
            }
            if (F::has(P, F_WIND_MIX) && (wmask & 7)) {            // (the plain gust's drag law is evaluated with the lanes' values packed, below)
                const V3 rel = v3(u.x - d.v.x, u.y - d.v.y, u.z - d.v.z);
                const float kn = P.k_wind * fast_sqrt(fmaf(rel.x, rel.x, fmaf(rel.y, rel.y, rel.z * rel.z)));
                Fwind = v3(kn * rel.x, kn * rel.y, kn * rel.z);
            }
            if (wmask & 8) {                                           // PAPER.md:204, episode time at the start of the step
                const float ph = P.wind_sine_omega * ((float)__float_as_uint(env4.w) * P.dt_c);
                float s1, c1;
                sincosf(ph, &s1, &c1);
                Fwind.x = fmaf(P.wind_sine_amp, s1, Fwind.x); Fwind.y = fmaf(P.wind_sine_amp, c1, Fwind.y);
                Fwind.z = fmaf(0.6f * P.wind_sine_amp, s1 * c1, Fwind.z);   // 0.3 sin 2x = 0.6 sin x cos x
            }
        }

        s.Fwind = Fwind; s.gust_out = gust_out;
        // Table 4 latency rows (Q51): this episode's delays in substeps from one Philox draw at the
        // episode's reset index.  The row issued at step t runs from substep d on: with d = (n - 1) K + r, 1 <= r <= K, substeps
        // k < r of this step run the row of n steps ago, the rest the row after it.  A controller decodes once, from the first.
        float4 a_first = act4, a_second = act4;
        int sw = -1, d_obs = 0;
        if (F::has(P, F_LAT)) {
            const uint32_t ep0 = __float_as_uint(env4.w);
            const uint4 lr = philox4x32_10(e + P.env_base, (uint32_t)jj, (t - 1u) - ep0, STREAM_LATENCY, P.seed_lo, P.seed_hi);
            d_obs = P.lat_s_lo + (int)(((lr.y >> 8) * (uint32_t)P.lat_s_n) >> 24);
            if (P.lat_a_n > 0) {
                const int d_act = P.lat_a_lo + (int)(((lr.x >> 8) * (uint32_t)P.lat_a_n) >> 24);
                float4 h0 = B.H0[drone], h1 = B.H1[drone], h2 = B.H2[drone];
                if (ep0 == 0u) h0 = h1 = h2 = act4;                    // primed with the episode's first row
                const int nb = (d_act + P.K - 1) / P.K, r = d_act - (nb - 1) * P.K;
                a_first = nb == 0 ? act4 : nb == 1 ? h0 : nb == 2 ? h1 : h2;
                a_second = nb <= 1 ? act4 : nb == 2 ? h0 : h1;
                const int at = F::act(P);
                if ((at == 0 || at == 3 || at == 4) && nb >= 1 && r < P.K) sw = r;
                if (active) { B.H2[drone] = h1; B.H1[drone] = h0; B.H0[drone] = act4; }
            }
        }
        s.sw = sw; s.d_obs = d_obs;
        // S1/S2 decode, S3 motor model (Eq.1-3); RPMs are held over the K substeps
        s.n_later[0] = s.n_later[1] = s.n_later[2] = s.n_later[3] = 0.0f;
        s.n[0] = s.n[1] = s.n[2] = s.n[3] = 0.0f;
        decode_front<FEAT>(P, a_first, d, s.n, s.mid);            // controller actions: the loops run on the lanes' values packed, below
        if (F::has(P, F_LAT) && s.sw >= 0) { DroneRegs dtmp = d; DecodeMid mtmp; decode_front<FEAT>(P, a_second, dtmp, s.n_later, mtmp); }   // direct rotor commands: stateless
        // Domain randomisation (Table 4): this episode's factors scale the true vehicle, not the controller's model above.
        // 1 / s_J is folded into the body torque (every stage torque is linear in it, the gyroscopic ratios do not change).
        s.kf_e = dr ? __fmul_rn(P.k_f, s.dr0.z) : P.k_f; s.kappa_e = dr ? __fmul_rn(P.kappa, __fdiv_rn(s.dr0.w, s.dr0.z)) : P.kappa;
        s.inv_sJ = dr ? __fdiv_rn(1.0f, s.dr0.y) : 1.0f; s.inv_m_e = dr ? __fdiv_rn(P.inv_m, s.dr0.x) : P.inv_m; s.g_e = dr ? __fmul_rn(P.g, s.dr1.w) : P.g;
        s.dwc_e = dr ? __fmul_rn(P.dw_coef, s.dr1.z) : P.dw_coef;
        s.nmax = dr ? __fmul_rn(P.max_rpm, s.dr3.y) : P.max_rpm;    // true motor saturation of this episode
        if (dr && !pid) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { s.n[i] = fminf(s.n[i], s.nmax); s.n_later[i] = fminf(s.n_later[i], s.nmax); }
        }
        // Table 4 motor lag (Q44): the rotors follow n through a first-order lag sampled exactly per substep
#pragma unroll
        for (int i = 0; i < 4; ++i) s.n_act[i] = s.n[i];
        s.lag_gain = 1.0f;
        if (lag) {
            const float4 r = B.N0[s.drone];
            s.n_act[0] = r.x; s.n_act[1] = r.y; s.n_act[2] = r.z; s.n_act[3] = r.w;
            s.lag_gain = 1.0f - __expf(-P.h / s.dr3.z);
        }
        s.hit = false;
        s.snap = sensed(d, v3(0, 0, 0));                              // sensor latency of a whole step: the state the step starts from
    }

    const bool flush = pending2 != 0xFFFFFFFFu;                  // two items wait: fence now, flags after the substeps
    if (flush) __threadfence();
    {   // the K substeps, state in registers: one drone per lane (float) or the lane's two drones as packed pairs (F2)
        const NPTag<NP> np;
        Slot& s0 = sl[0]; Slot& s1 = sl[NP - 1];
#define MDG_PK(f) pack_lanes(np, s0.f, s1.f)
        Body<T> bd;
        bd.p = v3t<T>(MDG_PK(d.p.x), MDG_PK(d.p.y), MDG_PK(d.p.z));
        bd.q.w = MDG_PK(d.q.w); bd.q.x = MDG_PK(d.q.x); bd.q.y = MDG_PK(d.q.y); bd.q.z = MDG_PK(d.q.z);
        bd.v = v3t<T>(MDG_PK(d.v.x), MDG_PK(d.v.y), MDG_PK(d.v.z));
        bd.w = v3t<T>(MDG_PK(d.w.x), MDG_PK(d.w.y), MDG_PK(d.w.z));
        T nn[4] = {MDG_PK(n[0]), MDG_PK(n[1]), MDG_PK(n[2]), MDG_PK(n[3])};
        if (pid) {                                                 // S2: position and attitude loops, mixer (control_loops)
            DecodeMidT<T> m;
            m.roll = MDG_PK(mid.roll); m.pitch = MDG_PK(mid.pitch); m.cpsi = MDG_PK(mid.cpsi); m.spsi = MDG_PK(mid.spsi);
            m.ncpsi = pack_lanes(np, -s0.mid.cpsi, -s1.mid.cpsi); m.nspsi = pack_lanes(np, -s0.mid.spsi, -s1.mid.spsi);
            m.e_p = v3t<T>(MDG_PK(mid.e_p.x), MDG_PK(mid.e_p.y), MDG_PK(mid.e_p.z));
            m.v_cmd = v3t<T>(MDG_PK(mid.v_cmd.x), MDG_PK(mid.v_cmd.y), MDG_PK(mid.v_cmd.z));
            m.e_psi = MDG_PK(mid.e_psi); m.thrust = MDG_PK(mid.T); m.phi_ref = MDG_PK(mid.phi_ref); m.th_ref = MDG_PK(mid.th_ref);
            V3T<T> Ip = v3t<T>(MDG_PK(d.Ip.x), MDG_PK(d.Ip.y), MDG_PK(d.Ip.z)), Ie = v3t<T>(MDG_PK(d.Ie.x), MDG_PK(d.Ie.y), MDG_PK(d.Ie.z));
            control_loops<FEAT>(P, m, bd.v, bd.w, Ip, Ie, nn);
            if (dr) {
                const T nmax = MDG_PK(nmax);
#pragma unroll
                for (int i = 0; i < 4; ++i) nn[i] = min_(nn[i], nmax);
            }
#pragma unroll
            for (int h = 0; h < NP; ++h) {
                sl[h].d.Ip = v3(half_of(Ip.x, h), half_of(Ip.y, h), half_of(Ip.z, h));
                sl[h].d.Ie = v3(half_of(Ie.x, h), half_of(Ie.y, h), half_of(Ie.z, h));
#pragma unroll
                for (int i = 0; i < 4; ++i) sl[h].n[i] = half_of(nn[i], h);
            }
        }
        // park what only the epilogue needs
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            const Slot& s = sl[h];
            float4* const st4 = stash0 + ((size_t)(wib * NP + h) * n_stash) * 32 + lane;
            st4[iIP * 32] = make_float4(0.0f, s.d.Ip.x, s.d.Ip.y, s.d.Ip.z);
            st4[iTG * 32] = s.tg;
            st4[iENV * 32] = s.env4;
            if (pid) st4[iIE * 32] = make_float4(s.d.Ie.x, s.d.Ie.y, s.d.Ie.z, 0.0f);
            if (F::act(P) == 1) st4[iSP * 32] = s.d.sp;
            if (obs_kin20) st4[iACT * 32] = s.act4;
        }
        asm volatile("" ::: "memory");                            // the epilogue re-reads them: no register copies kept across the loop

        if (F::has(P, F_WIND) && !F::has(P, F_WIND_MIX)) {        // PAPER.md:201 drag law on the gust just updated: F = k_w |u - v| (u - v) (Q28)
            const V3T<T> rel = v3t<T>(sub_(MDG_PK(env4.x), bd.v.x), sub_(MDG_PK(env4.y), bd.v.y), sub_(MDG_PK(env4.z), bd.v.z));
            const T kn = mul_(P.k_wind, sqrt_(dot3(rel, rel)));
            bd.a0 = v3t<T>(mul_(kn, rel.x), mul_(kn, rel.y), mul_(kn, rel.z));
        } else bd.a0 = v3t<T>(MDG_PK(Fwind.x), MDG_PK(Fwind.y), MDG_PK(Fwind.z));
        const T inv_m = MDG_PK(inv_m_e);                          // 1 / m folded into everything the substeps sum up
        bd.a0 = v3t<T>(fma_(bd.a0.x, inv_m, 0.0f), fma_(bd.a0.y, inv_m, 0.0f), fma_(bd.a0.z, inv_m, pack_lanes(np, -s0.g_e, -s1.g_e)));
        bd.ndwc = mul_(pack_lanes(np, -s0.dwc_e, -s1.dwc_e), inv_m);
        // S3 motor model (Eq.1-3) as a function of the rotor speeds: once per step, or every substep under the motor lag.  Every
        // product and sum is spelled out (mdg_dev.cuh: lane-generic arithmetic), so one env per lane and two round identically.
        auto motor_model = [&](const T (&nn)[4]) {
            const T kf = MDG_PK(kf_e);
            const T k0 = dr ? mul_(kf, MDG_PK(dr2.x)) : kf, k1 = dr ? mul_(kf, MDG_PK(dr2.y)) : kf,
                    k2 = dr ? mul_(kf, MDG_PK(dr2.z)) : kf, k3 = dr ? mul_(kf, MDG_PK(dr2.w)) : kf;
            // (products that are summed next are written as fma(a, b, 0): ptxas contracts a PACKED multiply-add pair into one FFMA2,
            //  which it never does for the scalar mul.rn / add.rn - see ang_acc_t)
            const T f0 = fma_(k0, mul_(nn[0], nn[0]), 0.0f), f1 = fma_(k1, mul_(nn[1], nn[1]), 0.0f), f2 = fma_(k2, mul_(nn[2], nn[2]), 0.0f),
                    f3 = fma_(k3, mul_(nn[3], nn[3]), 0.0f);
            const T f01 = add_(f0, f1), f23 = add_(f2, f3), f12 = add_(f1, f2), f03 = add_(f0, f3), f13 = add_(f1, f3), f02 = add_(f0, f2);
            const T thrust = add_(f01, f23);
            bd.thrust = fma_(thrust, inv_m, 0.0f);
            const T tz = mul_(MDG_PK(kappa_e), sub_(f13, f02));
            V3T<T> tau = F::has(P, F_CF2P) ? v3t<T>(mul_(P.arm, sub_(f1, f3)), mul_(P.arm, sub_(f2, f0)), tz)
                                            : v3t<T>(mul_(P.l, sub_(f01, f23)), mul_(P.l, sub_(f12, f03)), tz);
            if (dr) {
                const T isj = MDG_PK(inv_sJ), sxy = mul_(isj, MDG_PK(dr3.x));
                tau.x = mul_(tau.x, sxy); tau.y = mul_(tau.y, sxy); tau.z = mul_(tau.z, isj);
            }
            const T Om = mul_(P.rpm2rad, add_(add_(nn[0], nn[1]), add_(nn[2], nn[3])));
            bd.tau_b = tau;
            bd.k1_tau = v3t<T>(mul_(P.invJ[0], tau.x), mul_(P.invJ[1], tau.y), mul_(P.invJ[2], tau.z));
            const T cxy = dr ? mul_(mul_(-P.c_xy, MDG_PK(dr1.x)), Om) : mul_(-P.c_xy, Om);
            const T cz = dr ? fma_(mul_(-P.c_z, MDG_PK(dr1.x)), Om, 0.0f) : fma_(-P.c_z, Om, 0.0f);
            bd.gndT = dr ? mul_(mul_(P.gnd_coef, MDG_PK(dr1.y)), bd.thrust) : mul_(P.gnd_coef, bd.thrust);
            bd.cxy = fma_(cxy, inv_m, 0.0f);
            bd.dcz = mul_(sub_(cz, cxy), inv_m);
        };
        if (!lag) motor_model(nn);
        bool spun = false;                                         // two envs per lane: some substep was outside the series' range
#pragma unroll 1
        for (int k = 0; k < P.K; ++k) {
            if (NP == 1) {                                         // rotor commands that change inside the step: one env per lane only
                if (F::has(P, F_LAT) && s0.sw == k) {              // Q51: the next row arrives at this substep
#pragma unroll
                    for (int i = 0; i < 4; ++i) s0.n[i] = s0.n_later[i];
                    const T nn[4] = {MDG_PK(n[0]), MDG_PK(n[1]), MDG_PK(n[2]), MDG_PK(n[3])};
                    if (!lag) motor_model(nn);
                }
                if (lag) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) s0.n_act[i] = fmaf(s0.lag_gain, __fsub_rn(s0.n[i], s0.n_act[i]), s0.n_act[i]);
                    const T nn[4] = {MDG_PK(n_act[0]), MDG_PK(n_act[1]), MDG_PK(n_act[2]), MDG_PK(n_act[3])};
                    motor_model(nn);
                }
            }
            const SubstepFlags<T> fl = substep<G, FEAT, DEG>(P, bd, j, full_group);
            s0.hit |= half_of(fl.below, 0);
            if (NP == 2) { s1.hit |= half_of(fl.below, 1); spun |= any_(fl.fast); }
            if (NP == 1 && F::has(P, F_LAT) && k + 1 == P.K - s0.d_obs) {   // what the sensors report d_obs substeps later
                s0.snap.p = v3(half_of(bd.p.x, 0), half_of(bd.p.y, 0), half_of(bd.p.z, 0));
                s0.snap.v = v3(half_of(bd.v.x, 0), half_of(bd.v.y, 0), half_of(bd.v.z, 0));
                s0.snap.w = v3(half_of(bd.w.x, 0), half_of(bd.w.y, 0), half_of(bd.w.z, 0));
                s0.snap.q.w = half_of(bd.q.w, 0); s0.snap.q.x = half_of(bd.q.x, 0); s0.snap.q.y = half_of(bd.q.y, 0); s0.snap.q.z = half_of(bd.q.z, 0);
                s0.snap.eta = v3(0, 0, 0);
            }
        }
#undef MDG_PK
        if (NP == 2 && __any_sync(MDG_FULL, spun)) {               // rare: redo this item's substeps with the exact rotation path
            float r[2][13];
#pragma unroll
            for (int h = 0; h < NP; ++h) {
                Body<float> b1;
                b1.tau_b = half3(bd.tau_b, h); b1.k1_tau = half3(bd.k1_tau, h); b1.a0 = half3(bd.a0, h);
                b1.thrust = half_of(bd.thrust, h); b1.cxy = half_of(bd.cxy, h); b1.dcz = half_of(bd.dcz, h); b1.gndT = half_of(bd.gndT, h);
                b1.ndwc = half_of(bd.ndwc, h);
                const RedoOut o = redo_item_exact<G, FEAT, DEG>(P, B.P0 + sl[h].drone, B.P1 + sl[h].drone, B.P2 + sl[h].drone, B.P3 + sl[h].drone, b1, j, full_group);
                sl[h].hit = o.hit;
#pragma unroll
                for (int i = 0; i < 13; ++i) r[h][i] = o.s[i];
            }
            bd.p = v3t<T>(pack_lanes(np, r[0][0], r[NP - 1][0]), pack_lanes(np, r[0][1], r[NP - 1][1]), pack_lanes(np, r[0][2], r[NP - 1][2]));
            bd.q.w = pack_lanes(np, r[0][3], r[NP - 1][3]); bd.q.x = pack_lanes(np, r[0][4], r[NP - 1][4]);
            bd.q.y = pack_lanes(np, r[0][5], r[NP - 1][5]); bd.q.z = pack_lanes(np, r[0][6], r[NP - 1][6]);
            bd.v = v3t<T>(pack_lanes(np, r[0][7], r[NP - 1][7]), pack_lanes(np, r[0][8], r[NP - 1][8]), pack_lanes(np, r[0][9], r[NP - 1][9]));
            bd.w = v3t<T>(pack_lanes(np, r[0][10], r[NP - 1][10]), pack_lanes(np, r[0][11], r[NP - 1][11]), pack_lanes(np, r[0][12], r[NP - 1][12]));
        }
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            DroneRegs& d = sl[h].d;
            d.p = v3(half_of(bd.p.x, h), half_of(bd.p.y, h), half_of(bd.p.z, h));
            d.q.w = half_of(bd.q.w, h); d.q.x = half_of(bd.q.x, h); d.q.y = half_of(bd.q.y, h); d.q.z = half_of(bd.q.z, h);
            d.v = v3(half_of(bd.v.x, h), half_of(bd.v.y, h), half_of(bd.v.z, h));
            d.w = v3(half_of(bd.w.x, h), half_of(bd.w.y, h), half_of(bd.w.z, h));
        }
    }

    if (flush) { publish_flag(pending); publish_flag(pending2); pending = pending2 = 0xFFFFFFFFu; }
    const unsigned wt_after = take(drawn_l0);
    const unsigned probed_after = probe(wt_after);
#pragma unroll
    for (int h = 0; h < NP; ++h) {                                // back from the stash: controller memory, target, env word, action row
        Slot& s = sl[h];
        const float4* const st4 = stash0 + ((size_t)(wib * NP + h) * n_stash) * 32 + lane;
        const float4 f = st4[iIP * 32];
        s.d.Ip = v3(f.y, f.z, f.w);
        s.tg = st4[iTG * 32];
        s.env4 = st4[iENV * 32];
        if (pid) { const float4 i4 = st4[iIE * 32]; s.d.Ie = v3(i4.x, i4.y, i4.z); }
        if (F::act(P) == 1) s.d.sp = st4[iSP * 32];
        if (obs_kin20) s.act4 = st4[iACT * 32];
    }
#pragma unroll
    for (int h = 0; h < NP; ++h) {
        Slot& s = sl[h];
        DroneRegs& d = s.d;
        float4& env4 = s.env4;
        float4& tg = s.tg;
        const float4 act4 = s.act4;
        const unsigned e = s.e;
        const uint32_t t = s.t;
        const size_t drone = s.drone;
        const bool active = s.active, hit = s.hit;
        float (&n_act)[4] = s.n_act;
        const float4 gust_out = s.gust_out;
        const Sensed snap = s.snap;
        // S9-S11 epilogue on the end-of-step state
        const int gbase = lane & ~(G - 1);
        V3 eta = euler_zyx(d.q);
        V3 cen = v3(P.term_center[0], P.term_center[1], P.term_center[2]);
        const bool on_path = F::has(P, F_PATH);
        if (on_path) {                                                 // PAPER.md:325 (Q52): slots and the distance rule ride on the moving centre
            cen = path_centre(P, __float_as_uint(env4.w) + 1u);
            float sn, cs;
            sincospif(2.0f * (float)jj / (float)P.M, &sn, &cs);
            tg = make_float4(fmaf(P.form_radius, cs, cen.x), fmaf(P.form_radius, sn, cen.y), cen.z, tg.w);
        }
        const int term = F::term(P);
        const float aphi = fabsf(eta.x), ath = fabsf(eta.y);
        int flags = 0;                                                 // bit0 terminated, bit1 crash
        if (term == 1 || term == 3) { if (hit) flags |= 3; if (d.p.z > P.z_max) flags |= 1; }
        if (term != 0 && (aphi > P.term_tilt || ath > P.term_tilt)) flags |= 3;
        if (term == 2 || term == 3) {
            const float dx = d.p.x - cen.x, dy = d.p.y - cen.y, dz = d.p.z - cen.z;
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
        } else if (rew == 5) {                                         // FlyThroughAviary: capture handled below
            r = fmaf(P.wp_speed, fast_sqrt(fmaf(d.v.x, d.v.x, fmaf(d.v.y, d.v.y, d.v.z * d.v.z))),
                     fmaf(-P.wp_shaping, fast_sqrt(e2), -P.wp_omega * fast_sqrt(fmaf(d.w.x, d.w.x, fmaf(d.w.y, d.w.y, d.w.z * d.w.z)))));
        } else if (rew == 4) {                                         // VelocityAviary: target = (v*, omega_z*)
            const float ux = d.v.x - tg.x, uy = d.v.y - tg.y, uz = d.v.z - tg.z;
            const float u2 = fmaf(ux, ux, fmaf(uy, uy, uz * uz));
            r = -fast_sqrt(u2) - 0.1f * fabsf(d.w.z - tg.w) - 0.05f * (aphi + ath);
            if (u2 < P.at_target_radius2) r += 0.5f;
        } else {                                                       // formation: pair term below
            r = -fast_sqrt(e2);
        }
        // one pass over the env's drones serves the formation pair term and the adjacency row
        float adj[G];
    #pragma unroll
        for (int kk = 0; kk < G; ++kk) adj[kk] = 0.0f;
        const bool pairs = G > 1 && rew == 3;
        if (pairs || F::obs(P) == 1) {
            float pen = 0.0f;                                          // the self term is |0 - 0| = 0
    #pragma unroll
            for (int kk = 0; kk < G; ++kk) {
                const float ox = __shfl_sync(MDG_FULL, d.p.x, gbase + kk), oy = __shfl_sync(MDG_FULL, d.p.y, gbase + kk),
                            oz = __shfl_sync(MDG_FULL, d.p.z, gbase + kk);
                const float ax = d.p.x - ox, ay = d.p.y - oy, az = d.p.z - oz;
                const float d2 = fmaf(ax, ax, fmaf(ay, ay, az * az));
                adj[kk] = (kk == j || d2 < P.adj_radius2) ? 1.0f : 0.0f;
                if (pairs) {
                    float ddes;
                    if (F::has(P, F_TGT_CIRCLE)) ddes = P.chord[abs(j - kk)];
                    else {
                        const float ux = __shfl_sync(MDG_FULL, tg.x, gbase + kk), uy = __shfl_sync(MDG_FULL, tg.y, gbase + kk),
                                    uz = __shfl_sync(MDG_FULL, tg.z, gbase + kk);
                        const float bx = tg.x - ux, by = tg.y - uy, bz = tg.z - uz;
                        ddes = fast_sqrt(fmaf(bx, bx, fmaf(by, by, bz * bz)));
                    }
                    pen += (full_group || kk < P.M) ? fabsf(fast_sqrt(d2) - ddes) : 0.0f;
                }
            }
            if (pairs) r = fmaf(-0.25f, pen, r);                       // each unordered pair is seen from both ends
        }
        bool captured = false, last_wp = false;
        if (rew == 5) {
            captured = e2 < P.wp_radius2;
            last_wp = (int)tg.w + 1 >= P.wp_total;                     // running index over all laps
            if (captured) { r += P.wp_bonus; if (last_wp) flags |= 1; }   // the last capture ends the episode
        }
        const bool mine = full_group || j < P.M;
        const float rsum = group_sum<G>(mine ? r : 0.0f);
        const int gflags = group_or<G>(mine ? flags : 0);
        const uint32_t ep = __float_as_uint(env4.w) + 1u;
        const bool truncated = P.ep_steps > 0 && (int)ep >= P.ep_steps;
        const int done = (gflags & 1) | (truncated ? 2 : 0);
        uint32_t ep_out = ep;
        const bool do_reset = done != 0 && P.auto_reset != 0;
        float4 tg_out = tg;
        if (rew == 5 && captured && !last_wp) {                        // chase the next waypoint; its index rides in the 4th word
            const int kn = (int)tg.w + 1, kw = kn % P.n_waypoints;
            tg_out = make_float4(P.waypoints[3 * kw], P.waypoints[3 * kw + 1], P.waypoints[3 * kw + 2], (float)kn);
            if (active && !do_reset) B.P6[drone] = tg_out;
        }
        if (on_path && active && !do_reset) B.P6[drone] = tg_out;       // mdg_targets shows the slot of the moment
        if (__any_sync(MDG_FULL, do_reset)) {                          // S12 same-call auto-reset: rare, taken by the whole warp
            if (do_reset) {
                reset_drone(P, e, (uint32_t)jj, t, d, tg_out);
                if (F::has(P, F_DR)) {
                    float4 n0, n1, n2, n3;
                    draw_dr(P, e, (uint32_t)jj, t, n0, n1, n2, n3);
                    if (active) { B.R0[drone] = n0; B.R1[drone] = n1; B.R2[drone] = n2; B.R3[drone] = n3; }
                    if (lag) n_act[0] = n_act[1] = n_act[2] = n_act[3] = P.hover_rpm;
                }
                env4.x = env4.y = env4.z = 0.0f; ep_out = 0u;
                eta = euler_zyx(d.q);                                 // zeros unless Table 4's initial attitude range is on
                if (active) B.P6[drone] = tg_out;
            }
            if (F::obs(P) == 1) {                                      // the new episode's first observation
                float adj_new[G];
                adjacency<G>(P, d.p, lane, j, adj_new);
    #pragma unroll
                for (int kk = 0; kk < G; ++kk) adj[kk] = do_reset ? adj_new[kk] : adj[kk];
            }
        }
        if (active) {
            store_state(B, drone, d);
            if (pid) {
                B.P4[drone] = make_float4(d.Ie.x, d.Ie.y, d.Ie.z, 0.0f);
                if (F::act(P) == 1) B.P5[drone] = d.sp;
            }
            Sensed sn = sensed(d, eta);
            if (F::has(P, F_LAT) && !do_reset) { sn = snap; sn.eta = euler_zyx(snap.q); }   // a new episode's first row is its initial state
            if (F::has(P, F_SENS)) sense(P, e, (uint32_t)jj, t, ep_out, sn);   // Table 4 sensor rows: the stored state stays exact
            write_obs<G>(P, B.obs, drone, d, sn, adj, F::obs(P), do_reset ? make_float4(0, 0, 0, 0) : act4, tg_out);
            B.reward_d[drone] = r;
            if (lag) B.N0[drone] = make_float4(n_act[0], n_act[1], n_act[2], n_act[3]);
            if (j == 0) {
                env4.w = __uint_as_float(ep_out);
                B.E0[e] = env4; B.gstep[e] = t;
                B.reward[e] = rsum; B.done[e] = (uint8_t)done;
                if (F::has(P, F_WIND_MIX) && (P.wind_mask & 4) && F::has(P, F_WIND)) B.E1[e] = do_reset ? make_float4(0, 0, 0, 1.0f) : gust_out;
            }
        }
    }
    if (pending == 0xFFFFFFFFu) pending = wt; else pending2 = wt;
    if (wt_next >= n_items) break;
    wt = wt_next; wt_next = wt_after; probed_next = probed_after;
    }   // work-item loop
    __threadfence();
    publish_flag(pending);
    if (pending2 != 0xFFFFFFFFu) publish_flag(pending2);
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
    const int omode = (P.feat >> F_OBS_SHIFT) & 7;
    if (omode == 1) adjacency<G>(P, d.p, lane, j, adj);
    if (!active) return;
    store_state(B, drone, d);
    B.P4[drone] = make_float4(0, 0, 0, 0); B.P5[drone] = d.sp; B.P6[drone] = tg;
    float4 n0 = make_float4(1, 1, 1, 1), n1 = n0, n2 = n0, n3 = n0;
    if (P.feat & F_DR) draw_dr(P, e, (uint32_t)jj, 0u, n0, n1, n2, n3);
    B.R0[drone] = n0; B.R1[drone] = n1; B.R2[drone] = n2; B.R3[drone] = n3;
    B.N0[drone] = make_float4(P.hover_rpm, P.hover_rpm, P.hover_rpm, P.hover_rpm);
    Sensed sn = sensed(d, euler_zyx(d.q));
    if (P.feat & F_SENS) sense(P, e, (uint32_t)jj, 0u, 0u, sn);
    write_obs<G>(P, B.obs, drone, d, sn, adj, omode, make_float4(0, 0, 0, 0), tg);
    B.reward_d[drone] = 0.0f;
    if (j == 0) B.E1[e] = make_float4(0, 0, 0, 1.0f);
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
    const int omode = (P.feat >> F_OBS_SHIFT) & 7;
    if (omode == 1) adjacency<G>(P, d.p, lane, j, adj);
    if (!active) return;
    Sensed sn = sensed(d, euler_zyx(d.q));
    if (P.feat & F_SENS) sense(P, e, (uint32_t)jj, B.gstep[e], __float_as_uint(B.E0[e].w), sn);
    write_obs<G>(P, B.obs, drone, d, sn, adj, omode, make_float4(0, 0, 0, 0), B.P6[drone]);
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

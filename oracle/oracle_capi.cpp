// oracle/oracle_capi.cpp — TEST INFRASTRUCTURE: C entry points of the float64 CPU oracle
// (drone_oracle.hpp), loaded with ctypes by oracle/oracle.py.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / `--impl reference` legs may use it.  Shares nothing with the CUDA path.
#include <cstdio>
#include <cstdlib>
#include <string>
#include <thread>
// flop tally by phase of the control step: the oracle's header marks the phases, this file counts (drone_oracle.hpp: ORC_PHASE)
namespace orc { static thread_local int g_phase = 0; }
#define ORC_PHASE(k) (::orc::g_phase = (k))
#include "drone_oracle.hpp"
#include "camera_oracle.hpp"

namespace orc {

// Counting scalar: every add, sub, mul, div, compare and elementary function is one flop (an FMA is
// therefore two); negation, fabs and conversions are free.  SURVEY.md §8(d) counting rule.
static thread_local uint64_t g_flops = 0;
static thread_local uint64_t g_parts[PH_N] = {0};
#define ORC_TICK() (++g_flops, ++g_parts[g_phase])
struct Counted {
    double v;
    Counted() : v(0) {}
    Counted(double x) : v(x) {}
    explicit operator double() const { return v; }
    friend Counted operator+(const Counted& a, const Counted& b) { ORC_TICK(); return Counted(a.v + b.v); }
    friend Counted operator-(const Counted& a, const Counted& b) { ORC_TICK(); return Counted(a.v - b.v); }
    friend Counted operator*(const Counted& a, const Counted& b) { ORC_TICK(); return Counted(a.v * b.v); }
    friend Counted operator/(const Counted& a, const Counted& b) { ORC_TICK(); return Counted(a.v / b.v); }
    friend Counted operator-(const Counted& a) { return Counted(-a.v); }
    friend bool operator<(const Counted& a, const Counted& b) { ORC_TICK(); return a.v < b.v; }
    friend bool operator>(const Counted& a, const Counted& b) { ORC_TICK(); return a.v > b.v; }
};
inline Counted sqrt(const Counted& a) { ORC_TICK(); return Counted(std::sqrt(a.v)); }
inline Counted sin(const Counted& a) { ORC_TICK(); return Counted(std::sin(a.v)); }
inline Counted cos(const Counted& a) { ORC_TICK(); return Counted(std::cos(a.v)); }
inline Counted exp(const Counted& a) { ORC_TICK(); return Counted(std::exp(a.v)); }
inline Counted log(const Counted& a) { ORC_TICK(); return Counted(std::log(a.v)); }
inline Counted asin(const Counted& a) { ORC_TICK(); return Counted(std::asin(a.v)); }
inline Counted atan2(const Counted& a, const Counted& b) { ORC_TICK(); return Counted(std::atan2(a.v, b.v)); }
inline Counted fabs(const Counted& a) { return Counted(std::fabs(a.v)); }

static void run_threads(Sim& s, const float* actions, uint32_t t, int n_threads) {
    if (n_threads <= 1 || s.N < 2 * n_threads) { s.step_range<double>(0, s.N, actions, t); return; }
    std::vector<std::thread> th;
    const int chunk = (s.N + n_threads - 1) / n_threads;
    for (int i = 0; i < n_threads; ++i) {
        const int e0 = i * chunk, e1 = std::min(s.N, e0 + chunk);
        if (e0 >= e1) break;
        th.emplace_back([&s, e0, e1, actions, t] { s.step_range<double>(e0, e1, actions, t); });
    }
    for (auto& x : th) x.join();
}

struct Field { const char* name; int kind; size_t off; int len; };   // kind 0 double, 1 int
#define FD(n, len) {#n, 0, offsetof(Params, n), len}
#define FI(n) {#n, 1, offsetof(Params, n), 1}
static const Field FIELDS[] = {
    FD(m, 1), FD(g, 1), FD(L, 1), FD(k_f, 1), FD(k_m, 1), FD(J, 3), FD(r_p, 1), FD(tw_ratio, 1),
    FD(C_gnd, 1), FD(h_clip, 1), FD(c_xy, 1), FD(c_z, 1), FD(dw_C1, 1), FD(dw_C2, 1), FD(dw_C3, 1), FD(dw_dz_clip, 1),
    FD(k_wind, 1), FD(wind_sigma, 1), FD(wind_tau, 1), FI(sim_freq), FI(ctrl_freq), FI(aero_mask), FI(integrator),
    FD(Kp_pos, 3), FD(Ki_pos, 3), FD(Kd_pos, 3), FD(Kp_att, 3), FD(Ki_att, 3), FD(Kd_att, 3),
    FD(int_clamp_pos, 1), FD(int_clamp_att, 1), FI(dsl), FD(pos_rate_limit, 1), FD(yaw_rate_limit, 1), FD(a_ff, 3),
    FD(tilt_max, 1), FD(tau_xy_max, 1), FD(tau_z_max, 1), FI(obs_mode), FD(adj_radius, 1), FI(reward_mode),
    FD(at_target_radius, 1), FI(term_mode), FD(term_tilt, 1), FD(term_dist, 1), FD(term_center, 3), FD(z_max, 1),
    FD(episode_len_s, 1), FI(auto_reset), FI(reset_layout), FD(reset_center, 3), FD(reset_half, 3),
    FD(reset_z_lo, 1), FD(reset_z_hi, 1), FI(grid_cols), FD(grid_spacing, 1), FD(circle_radius, 1), FI(target_mode),
    FD(target_fixed, 3), FD(target_lo, 3), FD(target_hi, 3), FD(mh_z_lo, 1), FD(mh_z_hi, 1), FD(form_center, 3),
    FD(form_radius, 1), FI(env_index_base), FI(drone_model), FD(target_w_lo, 1), FD(target_w_hi, 1), FD(dr_alpha, 12), FD(reset_rpy_half, 3), FD(reset_vel_half, 3), FD(motor_lag_lo, 1), FD(motor_lag_hi, 1), FI(wind_mask), FD(wind_const, 3), FD(wind_sine_amp, 1), FD(wind_sine_omega, 1), FD(gust_prob, 1), FD(gust_max, 1), FD(gust_duration, 1), FI(n_waypoints), FD(waypoints, 24), FD(wp_radius, 1), FD(wp_bonus, 1), FD(wp_shaping, 1), FD(wp_speed, 1), FD(wp_omega, 1), FI(wp_laps), FD(obs_noise, 4), FD(obs_bias, 4), FD(dryden_airspeed, 1), FD(dryden_h_min, 1), FD(act_latency_lo, 1), FD(act_latency_hi, 1), FD(obs_latency_lo, 1), FD(obs_latency_hi, 1), FI(form_path_n), FD(form_path, 24), FD(form_speed, 1),
};
static const Field* find_field(const char* name) {
    for (const Field& f : FIELDS) if (std::string(f.name) == name) return &f;
    return nullptr;
}

}  // namespace orc

using namespace orc;

extern "C" {

void* orc_params_new(int model) { Params* p = new Params; default_params(model, *p); return p; }
void orc_params_free(void* p) { delete (Params*)p; }
int orc_params_set(void* p, const char* name, int idx, double value) {
    const Field* f = find_field(name);
    if (!f || idx < 0 || idx >= f->len) return -1;
    char* base = (char*)p + f->off;
    if (f->kind == 0) ((double*)base)[idx] = value; else ((int*)base)[idx] = (int)value;
    return 0;
}
int orc_params_get(const void* p, const char* name, int idx, double* value) {
    const Field* f = find_field(name);
    if (!f || idx < 0 || idx >= f->len) return -1;
    const char* base = (const char*)p + f->off;
    *value = f->kind == 0 ? ((const double*)base)[idx] : (double)((const int*)base)[idx];
    return 0;
}
// derived constants O1: out = [W, hover_rpm, max_rpm, l, kappa, s_max, h, dt_c, K, ep_steps, aero, integ]
void orc_derived(const void* p, int physics_mode, double* out) {
    const Derived d = derive(*(const Params*)p, physics_mode);
    const double v[12] = {d.W, d.hover_rpm, d.max_rpm, d.l, d.kappa, d.s_max, d.h, d.dt_c,
                          (double)d.K, (double)d.ep_steps, (double)d.aero, (double)d.integ};
    for (int i = 0; i < 12; ++i) out[i] = v[i];
}

void* orc_create(int n_envs, int n_drones, int physics_mode, int action_type, const void* params) {
    const Params& P = *(const Params*)params;
    if (n_envs < 1 || n_drones < 1 || P.ctrl_freq < 1 || P.sim_freq < P.ctrl_freq || P.sim_freq % P.ctrl_freq) return nullptr;
    const int K = P.sim_freq / P.ctrl_freq;                       // Q51: at most 3 control steps of action latency, 1 of sensor latency
    if (P.act_latency_lo < 0 || P.act_latency_hi < P.act_latency_lo || std::floor(P.act_latency_hi * P.sim_freq + 0.5) > 3 * K) return nullptr;
    if (P.obs_latency_lo < 0 || P.obs_latency_hi < P.obs_latency_lo || std::floor(P.obs_latency_hi * P.sim_freq + 0.5) > K) return nullptr;
    if (P.form_path_n < 0 || P.form_path_n > 8 || P.form_speed < 0) return nullptr;
    Sim* s = new Sim;
    s->init(n_envs, n_drones, physics_mode, action_type, P);
    return s;
}
void orc_destroy(void* h) { delete (Sim*)h; }
int orc_obs_dim(const void* h) { return ((const Sim*)h)->obs_dim(); }
void orc_reset(void* h, uint64_t seed) { ((Sim*)h)->reset_all(seed); }
void orc_step(void* h, const float* actions, int n_threads) {
    Sim& s = *(Sim*)h;
    const uint32_t t = s.gstep + 1;
    run_threads(s, actions, t, n_threads);
    s.gstep = t;
}
// algorithmic flops of one control step from the current state (the state is left untouched)
uint64_t orc_flop_tally(const void* h, const float* actions) {
    Sim copy = *(const Sim*)h;
    g_flops = 0;
    for (int k = 0; k < PH_N; ++k) g_parts[k] = 0;
    copy.step_range<Counted>(0, copy.N, actions, copy.gstep + 1);
    return g_flops;
}
// the same tally by phase (PH_* of drone_oracle.hpp: wind, decode, motor model, substep wrench, integrator, observation,
// reward + termination), filled by the last orc_flop_tally of this thread
void orc_flop_parts(uint64_t* out) { for (int k = 0; k < PH_N; ++k) out[k] = g_parts[k]; }
// flops of ONE call of a building block of the oracle on the counting scalar, on generic (non-degenerate) arguments:
// what tests/test_oracle_flop_tally.py compares with hand counts of the formulas
uint64_t orc_count_flops(const char* name) {
    Params P; default_params(MODEL_CF2X, P);
    const Derived D = derive(P, PHYS_MJC);
    Counted q[4] = {0.9, 0.1, -0.2, 0.3}, a3[3] = {0.3, -0.4, 0.5}, b3[3] = {0.7, 0.2, -0.6}, o3[3], o4[4], M[3][3];
    Counted b4[4] = {0.8, -0.3, 0.4, 0.1};
    const std::string n(name);
    g_flops = 0;
    if (n == "cross") cross(a3, b3, o3);
    else if (n == "mat_vec") { rotmat(q, M); g_flops = 0; mat_vec(M, a3, o3); }
    else if (n == "matT_vec") { rotmat(q, M); g_flops = 0; matT_vec(M, a3, o3); }
    else if (n == "rotmat") rotmat(q, M);
    else if (n == "quat_mul") quat_mul(q, b4, o4);
    else if (n == "quat_exp_step") quat_exp_step(q, a3, o4);
    else if (n == "quat_normalise") quat_normalise(q);
    else if (n == "euler_zyx") euler_zyx(q, o3);
    else if (n == "ang_acc") ang_acc(P, q, a3, b3, o3);
    else if (n == "motor_wrench") { Counted nn[4] = {14000.0, 14100.0, 14200.0, 14300.0}, T, tau[3], Om; motor_wrench(P, D, nn, T, tau, Om); }
    else if (n == "alloc_inverse") { Counted T = 0.26, s[4]; alloc_inverse(P, D, T, a3, s); }
    else if (n == "clampR_inside") { Counted x = 0.5; (void)clampR(x, 0.0, 1.0); }
    else if (n == "wrap_pi") { Counted x = 4.0; (void)wrap_pi(x); }
    else if (n == "integrate_rk4" || n == "integrate_euler") {
        Params P2 = P; P2.integrator = n == "integrate_rk4" ? INTEG_RK4 : INTEG_EULER;
        const Derived D2 = derive(P2, PHYS_MJC);
        Drone<Counted> d;
        for (int i = 0; i < 3; ++i) { d.p[i] = 1.0 + 0.1 * i; d.v[i] = 0.2 - 0.1 * i; d.w[i] = 0.5 + 0.3 * i; d.Fw[i] = 0.05 * (i + 1); d.tw[i] = 1e-4 * (i + 1); }
        for (int i = 0; i < 4; ++i) d.q[i] = q[i];
        for (int i = 0; i < DR_N; ++i) d.sc[i] = 1.0;
        d.hit = false; d.min_abs_pz = 1e30;
        quat_normalise(d.q);
        g_flops = 0;
        integrate(P2, D2, d);
    } else return ~0ull;
    return g_flops;
}

#define SIM ((Sim*)h)
void orc_get_state(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->state.data(), ((const Sim*)h)->state.size() * 8); }
void orc_set_state(void* h, const double* in) { std::memcpy(SIM->state.data(), in, SIM->state.size() * 8); }
void orc_get_pid(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->pid.data(), ((const Sim*)h)->pid.size() * 8); }
void orc_set_pid(void* h, const double* in) { std::memcpy(SIM->pid.data(), in, SIM->pid.size() * 8); }
void orc_get_targets(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->target.data(), ((const Sim*)h)->target.size() * 8); }
void orc_set_targets(void* h, const double* in) { std::memcpy(SIM->target.data(), in, SIM->target.size() * 8); }
void orc_get_wind(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->wind.data(), ((const Sim*)h)->wind.size() * 8); }
void orc_set_wind(void* h, const double* in) { std::memcpy(SIM->wind.data(), in, SIM->wind.size() * 8); }
void orc_get_dr(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->drs.data(), ((const Sim*)h)->drs.size() * 8); }
void orc_set_dr(void* h, const double* in) { std::memcpy(SIM->drs.data(), in, SIM->drs.size() * 8); }
void orc_get_ep_step(const void* h, uint32_t* out) { std::memcpy(out, ((const Sim*)h)->ep_step.data(), ((const Sim*)h)->ep_step.size() * 4); }
void orc_set_ep_step(void* h, const uint32_t* in) { std::memcpy(SIM->ep_step.data(), in, SIM->ep_step.size() * 4); }
uint32_t orc_get_gstep(const void* h) { return ((const Sim*)h)->gstep; }
void orc_get_rotor(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->rotor.data(), ((const Sim*)h)->rotor.size() * 8); }
void orc_set_rotor(void* h, const double* in) { std::memcpy(SIM->rotor.data(), in, SIM->rotor.size() * 8); }
void orc_get_gust(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->gust.data(), ((const Sim*)h)->gust.size() * 8); }
void orc_set_gust(void* h, const double* in) { std::memcpy(SIM->gust.data(), in, SIM->gust.size() * 8); }
void orc_get_reward_d(const void* h, double* out) { std::memcpy(out, ((const Sim*)h)->reward_d.data(), ((const Sim*)h)->reward_d.size() * 8); }
void orc_get_outputs(const void* h, double* obs, double* reward, uint8_t* done, double* margin) {
    const Sim& s = *(const Sim*)h;
    if (obs) std::memcpy(obs, s.obs.data(), s.obs.size() * 8);
    if (reward) std::memcpy(reward, s.reward.data(), s.reward.size() * 8);
    if (done) std::memcpy(done, s.done.data(), s.done.size());
    if (margin) std::memcpy(margin, s.margin.data(), s.margin.size() * 8);
}
// recompute obs of every env from the current state (after orc_set_state)
void orc_refresh_obs(void* h) {
    Sim& s = *SIM;
    std::vector<Drone<double>> buf(s.M);
    for (int e = 0; e < s.N; ++e) { double m; s.load(e, buf.data()); s.write_obs(e, buf.data(), m, s.gstep); s.margin[(size_t)e * 3 + 2] = m; }
}

// ---- probes used by the pins -------------------------------------------------------------------
// world-frame substep wrench of every drone of env e from the current state, for given rotor RPMs
// (wind force from the env's current wind state and the drones' current velocity when WIND is on)
void orc_probe_wrench(const void* h, int e, const double* rpm, double* F, double* tau) {
    const Sim& s = *(const Sim*)h;
    std::vector<Drone<double>> buf(s.M);
    s.load(e, buf.data());
    for (int i = 0; i < s.M; ++i) {
        Drone<double>& d = buf[i];
        for (int a = 0; a < 4; ++a) d.n[a] = rpm[i * 4 + a];
        motor_wrench(s.P, s.D, d.n, d.T, d.tau_b, d.Om, d.sc);
        if (s.D.aero & AERO_WIND) {
            double rel[3]; for (int a = 0; a < 3; ++a) rel[a] = s.wind[(size_t)e * 3 + a] - d.v[a];
            const double nr = std::sqrt(rel[0] * rel[0] + rel[1] * rel[1] + rel[2] * rel[2]);
            for (int a = 0; a < 3; ++a) d.Fwind[a] = s.P.k_wind * nr * rel[a];
        }
    }
    for (int i = 0; i < s.M; ++i) {
        substep_wrench(s.P, s.D, buf.data(), s.M, i);
        for (int a = 0; a < 3; ++a) { F[i * 3 + a] = buf[i].Fw[a]; tau[i * 3 + a] = buf[i].tw[a]; }
    }
}
// decode every drone's action into RPMs from the current state and PID memory; commit!=0 stores the
// updated PID memory
void orc_probe_decode(void* h, const float* actions, double* rpm, int commit) {
    Sim& s = *SIM;
    std::vector<Drone<double>> buf(s.M);
    for (int e = 0; e < s.N; ++e) {
        s.load(e, buf.data());
        for (int i = 0; i < s.M; ++i) {
            decode_action(s.P, s.D, s.action_type, actions + ((size_t)e * s.M + i) * 4, buf[i]);
            for (int a = 0; a < 4; ++a) rpm[((size_t)e * s.M + i) * 4 + a] = buf[i].n[a];
        }
        if (commit) s.store(e, buf.data());
    }
}
void orc_motor_wrench(const void* params, const double* rpm, double* out5) {   // T, tau xyz, Omega_sum
    const Params& P = *(const Params*)params; const Derived D = derive(P, 0);
    double T, tau[3], Om; motor_wrench(P, D, rpm, T, tau, Om);
    out5[0] = T; out5[1] = tau[0]; out5[2] = tau[1]; out5[3] = tau[2]; out5[4] = Om;
}
void orc_alloc_inverse(const void* params, double T, const double* tau, double* s4) {
    const Params& P = *(const Params*)params; const Derived D = derive(P, 0);
    alloc_inverse(*(const Params*)params, D, T, tau, s4);
}
void orc_euler_zyx(const double* q, double* eta) { euler_zyx(q, eta); }
void orc_quat_exp_step(const double* q, const double* phi, double* out) { quat_exp_step(q, phi, out); }
void orc_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t* out) {
    const PhiloxOut o = philox4x32_10(c0, c1, c2, c3, k0, k1);
    for (int i = 0; i < 4; ++i) out[i] = o.x[i];
}
// wind normals of env e at control step t, as O9 draws them
void orc_wind_normals(uint64_t seed, uint32_t e, uint32_t t, double* xi) {
    const PhiloxOut r = philox4x32_10(e, ENV_LEVEL, t, STREAM_WIND, (uint32_t)seed, (uint32_t)(seed >> 32));
    const double r1 = std::sqrt(-2.0 * std::log(1.0 - u01(r.x[0]))), r2 = std::sqrt(-2.0 * std::log(1.0 - u01(r.x[2])));
    xi[0] = r1 * std::cos(2.0 * PI * u01(r.x[1])); xi[1] = r1 * std::sin(2.0 * PI * u01(r.x[1]));
    xi[2] = r2 * std::cos(2.0 * PI * u01(r.x[3]));
}
// harness actions (stream 3): a[c] = base * fma(hi - lo, u_c, lo), every operation correctly rounded
// in fp32 so that the device generator can reproduce it bit for bit (last paragraph)
void orc_gen_actions(uint64_t seed, uint32_t t, int n_envs, int n_drones, float base, float lo, float hi, float* out, uint32_t env_base) {
    const float span = hi - lo;
    for (int e = 0; e < n_envs; ++e)
        for (int i = 0; i < n_drones; ++i) {
            const PhiloxOut r = philox4x32_10((uint32_t)e + env_base, (uint32_t)i, t, STREAM_ACTION, (uint32_t)seed, (uint32_t)(seed >> 32));
            for (int c = 0; c < 4; ++c) {
                const float u = (float)(r.x[c] >> 8) * (1.0f / 16777216.0f);
                const float f = std::fmaf(span, u, lo);
                out[((size_t)e * n_drones + i) * 4 + c] = base * f;
            }
        }
}

// NEXT-4 camera (camera_oracle.hpp).  state: [n_envs*n_drones][13] float64; cam: [H, W, fovy_deg, offset x y z, znear, zfar,
// body_a, body_c]; depth [D][H][W] float64, seg [D][H][W] u8, margin [D][H][W] float64 or NULL.
void orc_render_depth(const double* state, int n_envs, int n_drones, const double* cam, double* depth, uint8_t* seg,
                      double* margin, int n_threads) {
    CamParams cp;
    cp.H = (int)cam[0]; cp.W = (int)cam[1]; cp.fovy_deg = cam[2];
    cp.offset[0] = cam[3]; cp.offset[1] = cam[4]; cp.offset[2] = cam[5];
    cp.znear = cam[6]; cp.zfar = cam[7]; cp.body_a = cam[8]; cp.body_c = cam[9];
    const size_t px = (size_t)cp.H * cp.W;
    auto work = [&](int e0, int e1) {
        for (int e = e0; e < e1; ++e)
            for (int i = 0; i < n_drones; ++i) {
                const size_t d = (size_t)e * n_drones + i;
                render_camera(state + (size_t)e * n_drones * 13, n_drones, i, cp, depth + d * px, seg + d * px,
                              margin ? margin + d * px : nullptr);
            }
    };
    if (n_threads <= 1) { work(0, n_envs); return; }
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t)
        th.emplace_back(work, (int)((int64_t)n_envs * t / n_threads), (int)((int64_t)n_envs * (t + 1) / n_threads));
    for (auto& x : th) x.join();
}

// The same with the colour frame of reading Q53: rgba [D][H][W][4] u8, shade [D][H][W] float64 or NULL.
void orc_render_rgba(const double* state, int n_envs, int n_drones, const double* cam, double* depth, uint8_t* seg,
                     double* margin, uint8_t* rgba, double* shade, int n_threads) {
    CamParams cp;
    cp.H = (int)cam[0]; cp.W = (int)cam[1]; cp.fovy_deg = cam[2];
    cp.offset[0] = cam[3]; cp.offset[1] = cam[4]; cp.offset[2] = cam[5];
    cp.znear = cam[6]; cp.zfar = cam[7]; cp.body_a = cam[8]; cp.body_c = cam[9];
    const size_t px = (size_t)cp.H * cp.W;
    auto work = [&](int e0, int e1) {
        for (int e = e0; e < e1; ++e)
            for (int i = 0; i < n_drones; ++i) {
                const size_t d = (size_t)e * n_drones + i;
                render_camera(state + (size_t)e * n_drones * 13, n_drones, i, cp, depth + d * px, seg + d * px,
                              margin ? margin + d * px : nullptr, rgba + d * px * 4, shade ? shade + d * px : nullptr);
            }
    };
    if (n_threads <= 1) { work(0, n_envs); return; }
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t)
        th.emplace_back(work, (int)((int64_t)n_envs * t / n_threads), (int)((int64_t)n_envs * (t + 1) / n_threads));
    for (auto& x : th) x.join();
}
}  // extern "C"

// mdg.cu — host side of libmdg.so: the C ABI of include/mdg.h, the SoA allocator, parameter
// preprocessing, kernel dispatch and CUDA-graph replay.  No CPU fallback: every step runs in the
// kernels of mdg_kernels.cuh.
#include <mutex>
#include <nvrtc.h>
#include <nvtx3/nvToolsExt.h>
#include <dlfcn.h>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <tuple>
#include <vector>

#include "../../include/mdg.h"
#include "mdg_kernels.cuh"
#include "mdg_camera.cuh"

using namespace mdg;

static thread_local std::string g_err;
static int fail(int code, const std::string& msg) { g_err = msg; return code; }
#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t _e = (call);                                                                   \
        if (_e != cudaSuccess)                                                                     \
            return fail(_e == cudaErrorMemoryAllocation ? MDG_ENOMEM : MDG_ECUDA,                  \
                        std::string(#call) + ": " + cudaGetErrorString(_e));                       \
    } while (0)

typedef void (*step_fn)(const DevParams, const DevBuffers, const float4*);
typedef void (*aux_fn)(const DevParams, const DevBuffers);

struct mdg_env {
    int N, M, G, physics_mode, action_type;
    mdg_params hp;
    DevParams P;
    DevBuffers B;
    void* arena = nullptr;
    void* hist = nullptr;   // action-history planes H0..H2 (action latency only; outside the arena so that its layout never moves)
    size_t arena_bytes = 0;
    cudaStream_t stream = 0;
    cudaStream_t capture_stream = nullptr;
    step_fn step = nullptr;
    aux_fn reset = nullptr, refresh = nullptr;
    std::string kernel_name;
    int block = 128, max_blocks_per_sm = 0, smem = 0, minb = 4;
    int pdl = 1;
    int lanes = 1;                       // envs per lane group in the step kernel: 2 = packed FP32 pairs (grids that fill the device; MDG_LANES=1|2 forces)
    int jit = 1;                         // MDG_JIT=0: never compile at run time, use the generic kernel; MDG_JIT=require: fail instead of falling back
    std::string jit_note;                // why the run-time specialisation was not possible (empty: it was, or was not needed)
    bool saturating = false;             // the step grid occupies every resident block slot of the device
    uint32_t seq = 0;                    // step launches issued so far (kernel parameter: flags and dispenser parity, mdg_kernels.cuh)
    bool chainable = false;              // the last operation on this handle was a step (launched on last_stream, in capture last_capture)
    cudaStream_t last_stream = nullptr;
    unsigned long long last_capture = 0;
    float* stage = nullptr;              // device staging buffer of mdg_step_host (lazily allocated)
    cudaEvent_t order_event = nullptr;   // mdg_set_stream: orders the new stream behind work queued on the old one
    int n_sms = 0, step_grid = 0;        // persistent step kernel: one block per resident slot, looping over tiles
    int step_grid_chained = 0;           // grid of a launch that chains to the previous step (configure_launch)
    int64_t launches = 0;
    std::map<std::tuple<const void*, int, int64_t>, cudaGraphExec_t> graphs;
};

static int feature_word(const mdg_params& p, int physics_mode, int action_type, int M, int G) {
    int aero = 0, integ = MDG_INTEG_RK4;                  // Table 1
    switch (physics_mode) {
        case MDG_PHYS_MJC_GND: aero = MDG_AERO_GND; break;
        case MDG_PHYS_MJC_DRAG: aero = MDG_AERO_DRAG; break;
        case MDG_PHYS_MJC_DW: aero = MDG_AERO_DW; break;
        case MDG_PHYS_MJC_GND_DRAG_DW: aero = MDG_AERO_GND | MDG_AERO_DRAG | MDG_AERO_DW; break;
        case MDG_PHYS_DYN: integ = MDG_INTEG_EULER; break;
        default: break;
    }
    if (p.aero_mask >= 0) aero = p.aero_mask & 15;
    if (p.integrator >= 0) integ = p.integrator;
    int f = aero | (M == G ? F_FULL : 0);
    if (integ == MDG_INTEG_EULER) f |= F_EULER;
    f |= action_type << F_ACT_SHIFT;
    if (action_type == MDG_ACT_PID && p.dsl) f |= F_DSL;
    f |= p.obs_mode << F_OBS_SHIFT;
    if (p.drone_model == MDG_MODEL_CF2P) f |= F_CF2P;
    for (int i = 0; i < 12; ++i) if (p.dr_alpha[i] != 0.0f) f |= F_DR;
    if (p.motor_lag_hi > 0.0f) f |= F_DR | F_MLAG;
    if ((aero & MDG_AERO_WIND) && (p.wind_mask != MDG_WIND_DRYDEN || p.dryden_airspeed > 0.0f)) f |= F_WIND_MIX;
    for (int i = 0; i < 4; ++i) if (p.obs_noise[i] != 0.0f || p.obs_bias[i] != 0.0f) f |= F_SENS;
    if (p.act_latency_hi > 0.0f || p.obs_latency_hi > 0.0f) f |= F_LAT;
    if (p.target_mode == MDG_TGT_CIRCLE && p.form_path_n >= 2 && p.form_speed > 0.0f) f |= F_PATH;
    f |= p.reward_mode << F_REW_SHIFT;
    f |= p.term_mode << F_TERM_SHIFT;
    if (p.reward_mode == MDG_REW_FORMATION && p.target_mode == MDG_TGT_CIRCLE) f |= F_TGT_CIRCLE;
    if (p.J[0] == p.J[1]) f |= F_AXISYM;
    return f;
}

// host double -> device fp32 constants (O1 of DESIGN.md §2)
static void make_dev_params(const mdg_params& p, int N, int M, int feat, DevParams& D) {
    std::memset(&D, 0, sizeof(D));
    const double W = (double)p.m * p.g;
    const double hover2 = W / (4.0 * p.k_f);
    const double max_rpm = std::sqrt((double)p.tw_ratio * hover2);
    const double h = 1.0 / p.sim_freq, dtc = 1.0 / p.ctrl_freq;
    D.N = N; D.M = M; D.K = p.sim_freq / p.ctrl_freq;
    D.ep_steps = (int)std::llround((double)p.episode_len_s * p.ctrl_freq);
    D.auto_reset = p.auto_reset; D.feat = feat; D.env_base = p.env_index_base;
    D.reset_layout = p.reset_layout; D.target_mode = p.target_mode;
    D.grid_cols = p.grid_cols > 0 ? p.grid_cols : 1; D.grid_rows = (M + D.grid_cols - 1) / D.grid_cols;
    const int omode = (feat >> F_OBS_SHIFT) & 7;
    D.opd = omode == MDG_OBS_KIN20 ? 20 : omode == MDG_OBS_KIN12_TGT ? 16 : omode == MDG_OBS_KIN12_WP ? 18 : omode == MDG_OBS_KIN12_Z ? 13 : 12 + (omode == MDG_OBS_KIN12_ADJ ? M : 0);
    D.h = (float)h; D.half_h = (float)(0.5 * h); D.h_sixth = (float)(h / 6.0); D.half_h2 = (float)(0.5 * h * h);
    D.w2_exact[0] = (float)((0.28 / h) * (0.28 / h));      // degree-2 series: exact to 1e-7 up to |omega| h = 0.28 rad
    D.w2_exact[1] = (float)((0.75 / h) * (0.75 / h));      // degree-3 series: up to 0.75 rad
    for (int s = 0; s < 2; ++s) {                                  // Rodrigues series of R(c w)^T in y = |w|^2
        const double c = s ? h : 0.5 * h, c2 = c * c;
        float* A = s ? D.rotA_full : D.rotA_half; float* Bc = s ? D.rotB_full : D.rotB_half;
        A[0] = (float)c; A[1] = (float)(-c * c2 / 6.0); A[2] = (float)(c * c2 * c2 / 120.0); A[3] = (float)(-c * c2 * c2 * c2 / 5040.0);
        Bc[0] = (float)(c2 / 2.0); Bc[1] = (float)(-c2 * c2 / 24.0); Bc[2] = (float)(c2 * c2 * c2 / 720.0); Bc[3] = (float)(-c2 * c2 * c2 * c2 / 40320.0);
    }
    for (int i = 0; i < 4; ++i) { D.rotnA_half[i] = -D.rotA_half[i]; D.rotnA_full[i] = -D.rotA_full[i]; }
    {                                                             // Eq.7 increment for phi = (h/6) s in y = |s|^2
        const double c = h / 6.0, c2 = c * c;
        D.expC[0] = 1.0f; D.expC[1] = (float)(-c2 / 8.0); D.expC[2] = (float)(c2 * c2 / 384.0); D.expC[3] = (float)(-c2 * c2 * c2 / 46080.0);
        D.expS[0] = (float)(c / 2.0); D.expS[1] = (float)(-c * c2 / 48.0); D.expS[2] = (float)(c * c2 * c2 / 3840.0); D.expS[3] = (float)(-c * c2 * c2 * c2 / 645120.0);
    }
    {                                                             // the same for phi = h s (s = the RK4 mean of the stage rates)
        const double c = h, c2 = c * c;
        D.expCm[0] = 1.0f; D.expCm[1] = (float)(-c2 / 8.0); D.expCm[2] = (float)(c2 * c2 / 384.0); D.expCm[3] = (float)(-c2 * c2 * c2 / 46080.0);
        D.expSm[0] = (float)(c / 2.0); D.expSm[1] = (float)(-c * c2 / 48.0); D.expSm[2] = (float)(c * c2 * c2 / 3840.0); D.expSm[3] = (float)(-c * c2 * c2 * c2 / 645120.0);
    }
    D.inv_m = (float)(1.0 / p.m); D.g = p.g; D.m = p.m; D.inv_g = (float)(1.0 / p.g);
    for (int i = 0; i < 3; ++i) { D.J[i] = p.J[i]; D.invJ[i] = (float)(1.0 / p.J[i]); }
    D.gyro[0] = (float)(((double)p.J[2] - p.J[1]) / p.J[0]);
    D.gyro[1] = (float)(((double)p.J[0] - p.J[2]) / p.J[1]);
    D.gyro[2] = (float)(((double)p.J[1] - p.J[0]) / p.J[2]);
    for (int i = 0; i < 3; ++i) D.ngyro[i] = -D.gyro[i];
    const double l = p.L / std::sqrt(2.0), kappa = (double)p.k_m / p.k_f;
    D.k_f = p.k_f; D.inv_k_f = (float)(1.0 / p.k_f); D.l = (float)l; D.kappa = (float)kappa;
    D.inv_l = (float)(1.0 / l); D.inv_kappa = (float)(1.0 / kappa);
    D.max_rpm = (float)max_rpm; D.s_max = (float)(p.k_f * max_rpm * max_rpm); D.T_max = (float)(4.0 * p.k_f * max_rpm * max_rpm);
    D.rpm2rad = (float)(2.0 * M_PI / 60.0);
    D.hover_rpm = (float)std::sqrt(hover2); D.rpm_span = (float)(max_rpm - std::sqrt(hover2));
    D.arm = p.L; D.inv_arm = (float)(1.0 / p.L);
    D.gnd_coef = (float)((double)p.C_gnd * (p.r_p / 4.0) * (p.r_p / 4.0)); D.h_clip = p.h_clip;
    D.c_xy = p.c_xy; D.c_z = p.c_z;
    D.dw_coef = (float)((double)p.dw_C1 * (p.r_p / 4.0) * (p.r_p / 4.0)); D.dw_C2 = p.dw_C2; D.dw_C3 = p.dw_C3;
    D.dz_clip = p.dw_dz_clip; D.inv_dz_clip = p.dw_dz_clip > 0 ? (float)(1.0 / p.dw_dz_clip) : INFINITY;   // saturate(dz * inf) = [dz > 0]
    const double s2ln2 = std::sqrt(2.0 * std::log(2.0));
    D.dw_C2s = (float)(p.dw_C2 * s2ln2); D.dw_C3s = (float)(p.dw_C3 * s2ln2); D.dw_b2_min = (float)(2.0 * std::log(2.0) * 1e-12);
    D.dz_floor = p.dw_dz_clip > 1e-6f ? p.dw_dz_clip : 1e-6f;
    const double alpha = std::exp(-dtc / p.wind_tau);
    D.wind_alpha = (float)alpha; D.wind_gain = (float)(p.wind_sigma * std::sqrt(1.0 - alpha * alpha)); D.k_wind = p.k_wind;
    D.dryden_x = (float)(dtc * p.dryden_airspeed); D.dryden_h_min = p.dryden_h_min; D.wind_sigma = p.wind_sigma; D.inv_M = (float)(1.0 / M);
    D.gust_prob = p.gust_prob; D.gust_max = p.gust_max; D.gust_ds = (float)(dtc / p.gust_duration);
    D.wind_mask = p.wind_mask; D.wind_sine_amp = p.wind_sine_amp; D.wind_sine_omega = p.wind_sine_omega;
    for (int i = 0; i < 3; ++i) D.wind_const[i] = p.wind_const[i];
    D.dt_c = (float)dtc;
    for (int i = 0; i < 3; ++i) {
        D.Kp_pos[i] = p.Kp_pos[i]; D.Ki_pos[i] = p.Ki_pos[i]; D.Kd_pos[i] = p.Kd_pos[i];
        D.Kp_att[i] = p.Kp_att[i]; D.Ki_att[i] = p.Ki_att[i]; D.Kd_att[i] = p.Kd_att[i];
        D.a_ff[i] = p.a_ff[i]; D.term_center[i] = p.term_center[i];
        D.reset_center[i] = p.reset_center[i]; D.reset_half[i] = p.reset_half[i];
        D.target_fixed[i] = p.target_fixed[i]; D.target_lo[i] = p.target_lo[i]; D.target_hi[i] = p.target_hi[i];
        D.form_center[i] = p.form_center[i];
    }
    D.int_clamp_pos = p.int_clamp_pos; D.int_clamp_att = p.int_clamp_att;
    D.pos_step_max = (float)(p.pos_rate_limit * dtc); D.yaw_step_max = (float)(p.yaw_rate_limit * dtc);
    D.tilt_max = p.tilt_max; D.tau_xy_max = p.tau_xy_max; D.tau_z_max = p.tau_z_max;
    D.adj_radius2 = (float)((double)p.adj_radius * p.adj_radius); D.at_target_radius2 = (float)((double)p.at_target_radius * p.at_target_radius);
    D.term_tilt = p.term_tilt; D.term_dist2 = (float)((double)p.term_dist * p.term_dist); D.z_max = p.z_max;
    D.reset_z_lo = p.reset_z_lo; D.reset_z_hi = p.reset_z_hi; D.grid_spacing = p.grid_spacing; D.circle_radius = p.circle_radius;
    D.mh_z_lo = p.mh_z_lo; D.mh_z_hi = p.mh_z_hi; D.form_radius = p.form_radius;
    D.target_w_lo = p.target_w_lo; D.target_w_hi = p.target_w_hi;
    for (int i = 0; i < 12; ++i) D.dr_alpha[i] = p.dr_alpha[i];
    for (int i = 0; i < 3; ++i) { D.reset_rpy_half[i] = p.reset_rpy_half[i]; D.reset_vel_half[i] = p.reset_vel_half[i]; }
    D.motor_lag_lo = p.motor_lag_lo; D.motor_lag_hi = p.motor_lag_hi;
    D.sens_mask = 0u;
    for (int i = 0; i < 4; ++i) {
        D.obs_noise[i] = p.obs_noise[i]; D.obs_bias[i] = p.obs_bias[i];
        if (p.obs_noise[i] != 0.0f) D.sens_mask |= 1u;
        if (p.obs_bias[i] != 0.0f) D.sens_mask |= 2u;
    }
    D.path_n = p.form_path_n; D.path_rate = (float)(dtc * p.form_speed);
    {   // moving formation centre (Q52): side lengths and perimeter of the closed polygon, in double
        double per = 0.0;
        for (int k = 0; k < p.form_path_n && k < 8; ++k) {
            const int kn = (k + 1) % p.form_path_n;
            double l2 = 0.0;
            for (int a = 0; a < 3; ++a) { const double dlt = (double)p.form_path[3 * kn + a] - (double)p.form_path[3 * k + a]; l2 += dlt * dlt; }
            D.path_len[k] = (float)std::sqrt(l2); per += std::sqrt(l2);
        }
        D.path_perimeter = (float)per;
        for (int i = 0; i < 24; ++i) D.path[i] = p.form_path[i];
    }
    {   // Table 4 latency rows in substeps (Q51): uniform over round(lo f_sim) .. round(hi f_sim)
        const int a_lo = (int)std::floor((double)p.act_latency_lo * p.sim_freq + 0.5), a_hi = (int)std::floor((double)p.act_latency_hi * p.sim_freq + 0.5);
        const int s_lo = (int)std::floor((double)p.obs_latency_lo * p.sim_freq + 0.5), s_hi = (int)std::floor((double)p.obs_latency_hi * p.sim_freq + 0.5);
        D.lat_a_lo = a_lo; D.lat_a_n = p.act_latency_hi > 0.0f ? a_hi - a_lo + 1 : 0;
        D.lat_s_lo = s_lo; D.lat_s_n = p.obs_latency_hi > 0.0f ? s_hi - s_lo + 1 : 0;
    }
    D.wp_total = p.n_waypoints * p.wp_laps; D.wp_bonus = p.wp_bonus; D.wp_shaping = p.wp_shaping; D.wp_speed = p.wp_speed; D.wp_omega = p.wp_omega;
    D.n_waypoints = p.n_waypoints; D.wp_radius2 = (float)((double)p.wp_radius * p.wp_radius);
    for (int i = 0; i < 24; ++i) D.waypoints[i] = p.waypoints[i];
    for (int dlt = 0; dlt < 32; ++dlt) D.chord[dlt] = (float)(2.0 * p.form_radius * std::fabs(std::sin(M_PI * dlt / M)));
}

// ---- kernel dispatch: specialisations for the five benchmark configs, generic otherwise -------------
#define FEATW(aero, euler, act, dsl, adj, rew, term) \
    ((aero) | ((euler) ? F_EULER : 0) | ((act) << F_ACT_SHIFT) | ((dsl) ? F_DSL : 0) | ((adj) << F_OBS_SHIFT) | ((rew) << F_REW_SHIFT) | ((term) << F_TERM_SHIFT) | F_FULL | F_AXISYM)
static constexpr int FEAT_C1 = FEATW(0, 0, 0, 0, 0, 0, 1);
static constexpr int FEAT_C2 = FEATW(3, 0, 0, 0, 0, 0, 1);
static constexpr int FEAT_C3 = FEATW(0, 0, 1, 1, 0, 1, 2);
static constexpr int FEAT_C4 = FEATW(7, 0, 0, 0, 0, 2, 1);
static constexpr int FEAT_C5 = FEATW(15, 0, 2, 0, 1, 3, 3) | F_TGT_CIRCLE;

// Feature words whose substep loop can run two envs per lane as packed FP32 pairs (mdg_kernels.cuh): a compile-time word
// without rotor commands that change inside the step (motor lag, latency rows).
static constexpr bool lanes2_capable(int feat) { return feat >= 0 && !(feat & (F_MLAG | F_LAT)); }
// register budget variants of one specialisation: MINB resident 128-thread blocks per SM; lanes = envs per lane group (1 or 2)
template <int G, int FEAT> static step_fn pick_minb(int minb, int lanes) {
    if constexpr (lanes2_capable(FEAT)) {
        if (lanes == 2) return minb >= 4 ? step_kernel<G, FEAT, 4, 2> : step_kernel<G, FEAT, 3, 2>;
    }
    switch (minb) {
        case 5: return step_kernel<G, FEAT, 5, 1>;
        case 6: return step_kernel<G, FEAT, 6, 1>;
        case 7: return step_kernel<G, FEAT, 7, 1>;
        case 8: return step_kernel<G, FEAT, 8, 1>;
        default: return step_kernel<G, FEAT, 4, 1>;
    }
}

// ---- run-time specialisation: the handle's own feature word instantiated with NVRTC over the same source ---------------------
// A feature word without a precompiled specialisation would run the runtime-flag generic kernel at 1.7-2.1x the time
// (DESIGN.md 6).  Instead, step_kernel<G, FEAT, MINB> is compiled for exactly this word (about a second, cached per process);
// the sources are the .cuh files beside the library.  Any failure falls back to the generic kernel.  MDG_JIT=0 disables it.
extern "C" int mdg_version(void);
static std::map<std::tuple<int, int, int, int>, std::pair<step_fn, std::string>> g_jit;   // kernel or, on failure, why
static std::mutex g_jit_mutex;                                   // distinct handles may be created from different threads
static step_fn jit_step_kernel(int G, int feat, int minb, int lanes, std::string& why) {
    std::lock_guard<std::mutex> guard(g_jit_mutex);
    const auto key = std::make_tuple(G, feat, minb, lanes);
    auto it = g_jit.find(key);
    if (it != g_jit.end()) { why = it->second.second; return it->second.first; }   // a failed attempt is not repeated
    step_fn result = nullptr;
    auto done = [&](const std::string& msg) { why = msg; g_jit[key] = std::make_pair(result, msg); return result; };
    Dl_info info;
    if (!dladdr((void*)&mdg_version, &info) || !info.dli_fname) return done("dladdr cannot locate libmdg.so");
    std::string dir(info.dli_fname);
    const size_t slash = dir.find_last_of('/');
    dir = (slash == std::string::npos ? std::string(".") : dir.substr(0, slash)) + "/csrc";
    if (const char* ev = std::getenv("MDG_JIT_SRC")) dir = ev;   // where the .cuh sources are (default: csrc/ beside the library)
    const std::string src = "#include \"mdg_kernels.cuh\"\n";
    const char* hdr_names[2] = {"stdint.h", "cuda_runtime.h"};   // NVRTC has the CUDA built-ins; only the fixed-width names are missing
    const char* hdr_src[2] = {"#pragma once\ntypedef unsigned char uint8_t; typedef unsigned int uint32_t; typedef int int32_t; "
                              "typedef unsigned long long uint64_t; typedef long long int64_t; typedef unsigned long uintptr_t;\n",
                              "#pragma once\n"};
    nvrtcProgram prog = nullptr;
    if (nvrtcCreateProgram(&prog, src.c_str(), "mdg_jit.cu", 2, hdr_src, hdr_names) != NVRTC_SUCCESS) return done("nvrtcCreateProgram failed");
    const std::string expr = "mdg::step_kernel<" + std::to_string(G) + ", " + std::to_string(feat) + ", " + std::to_string(minb) + ", " + std::to_string(lanes) + ">";
    const std::string inc = "-I" + dir;
    const char* opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", inc.c_str()};
    std::vector<char> cubin;
    std::string msg;
    if (nvrtcAddNameExpression(prog, expr.c_str()) != NVRTC_SUCCESS) msg = "nvrtcAddNameExpression failed";
    else if (nvrtcCompileProgram(prog, 4, opts) != NVRTC_SUCCESS) {
        size_t ln = 0;
        std::string log;
        if (nvrtcGetProgramLogSize(prog, &ln) == NVRTC_SUCCESS && ln > 1) { log.resize(ln); nvrtcGetProgramLog(prog, &log[0]); }
        msg = "NVRTC could not compile " + expr + " from " + dir + ": " + log.substr(0, 300);
    } else {
        const char* lowered = nullptr;
        size_t nb = 0;
        if (nvrtcGetLoweredName(prog, expr.c_str(), &lowered) == NVRTC_SUCCESS && lowered && nvrtcGetCUBINSize(prog, &nb) == NVRTC_SUCCESS && nb > 0) {
            cubin.resize(nb);
            cudaLibrary_t lib = nullptr;
            cudaKernel_t kern = nullptr;
            if (nvrtcGetCUBIN(prog, cubin.data()) == NVRTC_SUCCESS &&
                cudaLibraryLoadData(&lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0) == cudaSuccess &&
                cudaLibraryGetKernel(&kern, lib, lowered) == cudaSuccess)
                result = reinterpret_cast<step_fn>(kern);       // kernel handles are accepted wherever the runtime takes a function pointer
            else { cudaGetLastError(); msg = "the compiled cubin could not be loaded (cudaLibraryLoadData / cudaLibraryGetKernel)"; }
        } else msg = "NVRTC produced no cubin";
    }
    nvrtcDestroyProgram(&prog);
    return done(msg);
}

static void pick_kernels(mdg_env* h) {
    const int f = h->P.feat;
    h->step = nullptr;
    if (h->lanes == 2 && !lanes2_capable(f)) h->lanes = 1;
    const int mb2 = h->minb >= 4 ? 4 : 3;                            // two envs per lane: 128 or 168 registers
#define SPECIAL(g, fw, name) if (h->G == (g) && f == (fw)) { h->step = pick_minb<(g), (fw)>(h->minb, h->lanes); h->kernel_name = name; }
    SPECIAL(1, FEAT_C1, "step_kernel<G=1,rigid,rpm,hover>")
    SPECIAL(1, FEATW(0, 0, 3, 0, 0, 0, 1), "step_kernel<G=1,rigid,rpm_norm,hover>")   // the paper's own MJX workload
    SPECIAL(1, FEAT_C2, "step_kernel<G=1,gnd+drag,rpm,hover>")
    SPECIAL(1, FEAT_C3, "step_kernel<G=1,rigid,pid+dsl,negsqdist>")
    SPECIAL(8, FEAT_C4, "step_kernel<G=8,gnd+drag+dw,rpm,multihover>")
    SPECIAL(4, FEAT_C5, "step_kernel<G=4,gnd+drag+dw+wind,vel,adj,formation>")
    SPECIAL(4, FEAT_C5 | F_EULER, "step_kernel<G=4,gnd+drag+dw+wind,vel,adj,formation,dyn>")   // Table 1's DYN integrator on the metric's config
    SPECIAL(4, FEAT_C5 | F_DR | F_MLAG | F_SENS | F_LAT, "step_kernel<G=4,gnd+drag+dw+wind,vel,adj,formation,table4>")   // every row of Table 4 on it
#undef SPECIAL
    h->jit_note.clear();
    if (!h->step && h->jit) {                                        // no precompiled specialisation: instantiate this word now
        const int mb = h->lanes == 2 ? mb2 : (h->minb < 4 ? 4 : (h->minb > 8 ? 8 : h->minb));
        h->step = jit_step_kernel(h->G, f, mb, h->lanes, h->jit_note);
        if (h->step) h->kernel_name = "step_kernel<G=" + std::to_string(h->G) + ",jit:" + std::to_string(f) + ">";
    }
    if (!h->step) h->lanes = 1;                                      // the runtime-flag kernel: one env per lane
    if (h->step && h->lanes == 2) h->kernel_name.insert(h->kernel_name.size() - 1, ",x2");   // two envs per lane, packed FP32 pairs
#define GENERIC(g) case g: if (!h->step) { h->step = h->minb <= 3 ? step_kernel<g, -1, 3, 1> : step_kernel<g, -1, 4, 1>; h->kernel_name = "step_kernel<G=" #g ",generic>"; } \
                   h->reset = reset_kernel<g>; h->refresh = refresh_obs_kernel<g>; break;
    switch (h->G) { GENERIC(1) GENERIC(2) GENERIC(4) GENERIC(8) GENERIC(16) GENERIC(32) }
#undef GENERIC
}

// ---- helpers --------------------------------------------------------------------------------------
static int configure_launch(mdg_env* h) {
    h->P.zero = 0u;
    const int act_t = (h->P.feat >> F_ACT_SHIFT) & 7, obs_t = (h->P.feat >> F_OBS_SHIFT) & 7;
    const int n_stash = 3 + ((act_t == 1 || act_t == 2 || act_t == 5) ? 1 : 0) + (act_t == 1 ? 1 : 0) + (obs_t == 2 ? 1 : 0);   // as the kernel counts them
    const int stage_bytes = (h->block / 32) * h->lanes * ((int)sizeof(WarpStage) + n_stash * 512);   // landing zone + stash per warp and env slot
    h->smem = stage_bytes;
    if (h->max_blocks_per_sm > 0) {          // cap residency by padding the dynamic shared-memory request
        int s = (228 * 1024) / h->max_blocks_per_sm - 1024;
        if (s > 227 * 1024) s = 227 * 1024;
        if ((s & ~127) > h->smem) h->smem = s & ~127;
    }
    CU(cudaFuncSetAttribute((const void*)h->step, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem > 48 * 1024 ? h->smem : 48 * 1024));
    if (!h->n_sms) {
        int dev = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&h->n_sms, cudaDevAttrMultiProcessorCount, dev));
    }
    int resident = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, (const void*)h->step, h->block, h->smem));
    if (resident < 1) return fail(MDG_ECUDA, "configure_launch: the step kernel does not fit on an SM");
    const long long epw = (long long)h->lanes * (32 / h->G), wpb = h->block / 32;   // envs per work item (one warp), warps per block
    const long long items = ((long long)h->N + epw - 1) / epw, blocks = (items + wpb - 1) / wpb;
    const long long slots = (long long)h->n_sms * resident;
    h->step_grid = (int)(blocks < slots ? blocks : slots);
    // A launch that chains to the previous step shares the device with its neighbours in the stream anyway, so it need not
    // bring a block for every slot: with one block per SM fewer (two envs per lane, four resident blocks) every warp handles
    // more items per launch and pays its start-up and final fence less often, and the free slots are taken by the next
    // launch's blocks (same-box A/B on config 5: 19.04 -> 18.63 us per step in the first 40 ms, 19.3 -> 19.1 once the power cap
    // bites; its DYN variant 16.0 -> 15.2 and 16.4 -> 16.1; no gain with one env per lane, a 1 % loss when a warp has seven
    // items per launch anyway).  A launch that waits for the whole stream (mdg_step) keeps the full grid.
    h->step_grid_chained = h->step_grid;
    if (h->lanes == 2 && resident >= 4 && items >= slots * wpb && items < 3 * slots * wpb) h->step_grid_chained = h->n_sms * (resident - 1);
    // Item-level chaining of consecutive steps.  A grid that fills every resident slot gives each warp the item of its own
    // index first and hands the others out through a ticket dispenser (which therefore needs items >= warps); four dispensers
    // take turns, which needs "at most four step kernels of a handle in flight": a successor's blocks can only start in free
    // slots, and its own successor only once all of those have started, so for a fifth launch to draw from a dispenser a warp
    // of the first is still using, three whole grids would have to start and largely finish while that warp stalls.  A smaller grid gives every warp exactly one item (its index), draws
    // nothing, and may therefore be chained to any depth.
    h->saturating = items >= slots * wpb;
    h->P.static_items = h->saturating ? 0u : 1u;                   // one warp per item, no dispenser: any depth of chained launches is safe
    return MDG_OK;
}
static inline unsigned grid_for(const mdg_env* h, int block) {
    const size_t threads = (size_t)h->N * h->G;
    return (unsigned)((threads + block - 1) / block);
}
static void drop_graphs(mdg_env* h) {
    for (auto& kv : h->graphs) cudaGraphExecDestroy(kv.second);
    h->graphs.clear();
}
// One launch of the fused step.  want_chain: the caller vouches that the actions were complete before the previous step of this
// handle was enqueued (mdg_step_chained, the inner launches of mdg_step_many); the kernel then skips the grid-wide wait behind
// the previous kernel of the stream and orders itself item by item behind the previous step (mdg_kernels.cuh) - but only if that
// previous step really is the previous operation of this handle, on this stream and in the same capture (or both outside one).
static int launch_step(mdg_env* h, const float* actions_dev, cudaStream_t s, bool want_chain) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    unsigned long long cap_id = 0;
    CU(cudaStreamGetCaptureInfo(s, &cap, &cap_id));
    if (cap != cudaStreamCaptureStatusActive) cap_id = 0;
    h->seq += 1;
    h->P.seq = h->seq;
    h->P.chain = (want_chain && h->pdl && h->chainable && h->last_stream == s && h->last_capture == cap_id) ? 1u : 0u;
    h->chainable = true; h->last_stream = s; h->last_capture = cap_id;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(h->P.chain ? h->step_grid_chained : h->step_grid)); cfg.blockDim = dim3((unsigned)h->block);
    cfg.dynamicSmemBytes = (size_t)h->smem; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = h->pdl ? 1 : 0;
    nvtxRangePushA("mdg_step");                                     // visible in Nsight timelines, free without a tool attached
    const cudaError_t ce = cudaLaunchKernelEx(&cfg, h->step, h->P, h->B, reinterpret_cast<const float4*>(actions_dev));
    nvtxRangePop();
    if (ce != cudaSuccess) { h->chainable = false; return fail(MDG_ECUDA, std::string("cudaLaunchKernelEx(step_kernel): ") + cudaGetErrorString(ce)); }
    h->launches += 1;
    return MDG_OK;
}

extern "C" {

int mdg_version(void) { return 100; }
const char* mdg_last_error(void) { return g_err.c_str(); }

int mdg_default_params(int drone_model, mdg_params* p) {
    if (!p) return fail(MDG_EINVAL, "mdg_default_params: out is NULL");
    if (drone_model != MDG_MODEL_CF2X && drone_model != MDG_MODEL_CF2P && drone_model != MDG_MODEL_RACE)
        return fail(MDG_EINVAL, "mdg_default_params: unknown drone model");
    std::memset(p, 0, sizeof(*p));
    p->struct_size = (uint32_t)sizeof(mdg_params);
    p->drone_model = drone_model;
    if (drone_model == MDG_MODEL_RACE) {     // Table 2, RACE column
        p->m = 0.250f; p->L = 0.125f; p->tw_ratio = 4.0f; p->J[0] = p->J[1] = 4.86e-4f; p->J[2] = 8.80e-4f;
        p->k_f = 1.28e-8f; p->k_m = 5.96e-10f; p->r_p = 0.0635f;
    } else {                                 // Table 2, CF2X column
        p->m = 0.027f; p->L = 0.0397f; p->tw_ratio = 2.25f; p->J[0] = p->J[1] = 1.4e-5f; p->J[2] = 2.17e-5f;
        p->k_f = 3.16e-10f; p->k_m = 7.94e-12f; p->r_p = 0.02325f;
    }
    p->g = 9.81f;
    p->C_gnd = 11.36859f; p->c_xy = 9.1785e-7f; p->c_z = 10.311e-7f;
    p->h_clip = (float)(0.25 * p->r_p * std::sqrt(15.0 * p->C_gnd / 4.0));
    p->dw_C1 = 2267.18f; p->dw_C2 = 0.16f; p->dw_C3 = -0.11f; p->dw_dz_clip = 0.1f;
    p->k_wind = 0.5f * 1.225f * 1.0f * 0.01f; p->wind_sigma = 0.5f; p->wind_tau = 1.0f;
    p->wind_mask = MDG_WIND_DRYDEN; p->wind_sine_omega = (float)M_PI;
    p->gust_prob = 0.02f; p->gust_max = 1.0f; p->gust_duration = 0.5f;
    const float wps[15] = {0, 0, 1, 1, 0, 1, 1, 1, 1.5f, 0, 1, 1, 0, 0, 0.5f};          // PAPER.md:321 default list
    p->n_waypoints = 5; for (int i = 0; i < 15; ++i) p->waypoints[i] = wps[i];
    p->wp_radius = 0.1f; p->wp_bonus = 10.0f; p->wp_shaping = 0.1f; p->wp_speed = 0.0f; p->wp_omega = 0.01f; p->wp_laps = 1;
    p->dryden_airspeed = 0.0f; p->dryden_h_min = 0.05f;
    p->sim_freq = 240; p->ctrl_freq = 48;
    p->aero_mask = -1; p->integrator = -1;
    const float kp[3] = {0.4f, 0.4f, 1.0f}, ki[3] = {0.01f, 0.01f, 0.01f}, kd[3] = {0.9f, 0.9f, 2.0f};   // Table 6
    const float ap[3] = {2e-3f, 2e-3f, 1e-3f}, ai[3] = {0, 0, 1e-4f}, ad[3] = {5e-4f, 5e-4f, 2e-4f};
    for (int i = 0; i < 3; ++i) {
        p->Kp_pos[i] = kp[i]; p->Ki_pos[i] = ki[i]; p->Kd_pos[i] = kd[i];
        p->Kp_att[i] = ap[i]; p->Ki_att[i] = ai[i]; p->Kd_att[i] = ad[i];
    }
    p->int_clamp_pos = 2.0f; p->int_clamp_att = 0.5f; p->dsl = 0;
    p->pos_rate_limit = 2.0f; p->yaw_rate_limit = (float)M_PI; p->tilt_max = 0.5f;
    const double s_hover = (double)p->m * p->g / 4.0;
    p->tau_xy_max = (float)(4.0 * (p->L / std::sqrt(2.0)) * s_hover / 3.0);
    if (drone_model == MDG_MODEL_CF2P) p->tau_xy_max = (float)(2.0 * p->L * s_hover / 3.0);   // two rotors per axis, same rule
    p->tau_z_max = (float)(4.0 * ((double)p->k_m / p->k_f) * s_hover / 3.0);
    p->obs_mode = MDG_OBS_KIN12; p->adj_radius = 0.5f;
    p->reward_mode = MDG_REW_HOVER; p->at_target_radius = 0.05f;
    p->term_mode = MDG_TERM_HOVER; p->term_tilt = (float)(M_PI / 2); p->term_dist = 3.0f; p->z_max = 3.0f;
    p->episode_len_s = 10.0f; p->auto_reset = 1;
    p->reset_layout = MDG_LAYOUT_NONE; p->reset_center[2] = 1.0f;
    p->reset_half[0] = p->reset_half[1] = p->reset_half[2] = 0.1f;
    p->grid_cols = 4; p->grid_spacing = 0.3f; p->circle_radius = 0.3f;
    p->target_mode = MDG_TGT_FIXED; p->target_fixed[2] = 1.0f;
    p->target_lo[0] = p->target_lo[1] = -1.0f; p->target_lo[2] = 0.2f;
    p->target_hi[0] = p->target_hi[1] = 1.0f; p->target_hi[2] = 2.0f;
    p->mh_z_lo = 0.7f; p->mh_z_hi = 1.2f; p->form_center[2] = 1.0f; p->form_radius = 0.3f;
    return MDG_OK;
}

int mdg_create(int n_envs, int n_drones, int physics_mode, int action_type, const mdg_params* params, mdg_env** out) {
    if (!out) return fail(MDG_EINVAL, "mdg_create: out is NULL");
    *out = nullptr;
    mdg_params p;
    if (params) {
        if (params->struct_size != sizeof(mdg_params)) return fail(MDG_EINVAL, "mdg_create: params->struct_size mismatch");
        p = *params;
    } else mdg_default_params(MDG_MODEL_CF2X, &p);
    if (n_envs < 1 || n_drones < 1 || n_drones > 32) return fail(MDG_EINVAL, "mdg_create: need n_envs >= 1 and 1 <= n_drones <= 32");
    if ((int64_t)n_envs * 32 > (int64_t)1 << 31) return fail(MDG_EINVAL, "mdg_create: n_envs too large");
    if (physics_mode < 0 || physics_mode > MDG_PHYS_DYN) return fail(MDG_EINVAL, "mdg_create: unknown physics_mode");
    if (action_type < 0 || action_type > MDG_ACT_ATTITUDE) return fail(MDG_EINVAL, "mdg_create: unknown action_type");
    if (p.ctrl_freq < 1 || p.sim_freq < p.ctrl_freq || p.sim_freq % p.ctrl_freq)
        return fail(MDG_EINVAL, "mdg_create: sim_freq must be a positive integer multiple of ctrl_freq (PAPER.md:169)");
    if (p.obs_mode < 0 || p.obs_mode > 5 || p.n_waypoints < 0 || p.n_waypoints > 8 || p.motor_lag_lo < 0 || p.motor_lag_hi < p.motor_lag_lo || p.wp_laps < 0 || (p.wind_mask & ~15) || !(p.gust_duration > 0) || p.drone_model < 0 || p.drone_model > 2 || p.reward_mode < 0 || p.reward_mode > 5 || p.term_mode < 0 || p.term_mode > 3 ||
        p.reset_layout < 0 || p.reset_layout > 2 || p.target_mode < 0 || p.target_mode > 4 || p.integrator > 1 || p.aero_mask > 15)
        return fail(MDG_EINVAL, "mdg_create: enum field out of range in params");
    {
        const int Ks = p.sim_freq / p.ctrl_freq;
        if (!(p.act_latency_lo >= 0) || !(p.act_latency_hi >= p.act_latency_lo) || std::floor((double)p.act_latency_hi * p.sim_freq + 0.5) > 3 * Ks)
            return fail(MDG_EINVAL, "mdg_create: action latency must satisfy 0 <= lo <= hi <= 3 control steps");
        if (!(p.obs_latency_lo >= 0) || !(p.obs_latency_hi >= p.obs_latency_lo) || std::floor((double)p.obs_latency_hi * p.sim_freq + 0.5) > Ks)
            return fail(MDG_EINVAL, "mdg_create: sensor latency must satisfy 0 <= lo <= hi <= 1 control step");
    }
    if (p.form_path_n < 0 || p.form_path_n > 8 || !(p.form_speed >= 0)) return fail(MDG_EINVAL, "mdg_create: form_path_n in [0, 8], form_speed >= 0");
    if (!(p.dryden_airspeed >= 0) || (p.dryden_airspeed > 0 && !(p.dryden_h_min > 0)))
        return fail(MDG_EINVAL, "mdg_create: dryden_airspeed must be >= 0 and dryden_h_min > 0");
    for (int i = 0; i < 4; ++i)
        if (!(p.obs_noise[i] >= 0) || !(p.obs_bias[i] >= 0)) return fail(MDG_EINVAL, "mdg_create: obs_noise / obs_bias must be >= 0");
    if (!(p.m > 0) || !(p.k_f > 0) || !(p.k_m > 0) || !(p.J[0] > 0) || !(p.J[1] > 0) || !(p.J[2] > 0) || !(p.g > 0) || !(p.wind_tau > 0))
        return fail(MDG_EINVAL, "mdg_create: m, g, k_f, k_m, J, wind_tau must be positive");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(MDG_ECUDA, "mdg_create: no CUDA device (this library has no CPU fallback)");
    }
    mdg_env* h = new mdg_env;
    h->N = n_envs; h->M = n_drones; h->physics_mode = physics_mode; h->action_type = action_type; h->hp = p;
    int G = 1; while (G < n_drones) G <<= 1;
    h->G = G;
    if (const char* ev = std::getenv("MDG_PDL")) h->pdl = ev[0] != '0';
    if (const char* ev = std::getenv("MDG_JIT")) h->jit = ev[0] == '0' ? 0 : (ev[0] == 'r' ? 2 : 1);   // 0: generic kernel only; require: no silent fallback
    make_dev_params(p, n_envs, n_drones, feature_word(p, physics_mode, action_type, n_drones, G), h->P);
    pick_kernels(h);
    // one arena: 7 drone planes, env plane, gstep, obs, reward, done (each 256 B aligned)
    const size_t D = (size_t)n_envs * n_drones;
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t plane = al(D * sizeof(float4)), eplane = al((size_t)n_envs * sizeof(float4)), gs = al((size_t)n_envs * 4),
                 ob = al(D * h->P.opd * sizeof(float)), rw = al((size_t)n_envs * 4), dn = al((size_t)n_envs);
    const size_t n_items_max = (size_t)n_envs;                     // >= work items for any G
    const size_t rd = al(D * sizeof(float));
    // The first 2 MiB of the allocation stay unused: the latency-bound configs ran 30-45 % slower (config 4: 9.3 vs 6.6 us
    // per step) with the buffers at the very start of the cudaMalloc block - measured, mechanism not identified.
    const size_t front_pad = (size_t)2 << 20;
    h->arena_bytes = front_pad + rd + 12 * plane + 2 * eplane + gs + ob + rw + dn + 256 + al(n_items_max * 4);
    cudaError_t ce = cudaMalloc(&h->arena, h->arena_bytes);
    if (ce != cudaSuccess) { delete h; return fail(MDG_ENOMEM, std::string("mdg_create: cudaMalloc: ") + cudaGetErrorString(ce)); }
    ce = cudaMemset(h->arena, 0, h->arena_bytes);
    if (ce != cudaSuccess) { cudaFree(h->arena); delete h; return fail(MDG_ECUDA, std::string("mdg_create: cudaMemset: ") + cudaGetErrorString(ce)); }
    char* c = (char*)h->arena + front_pad;
    float4** planes[12] = {&h->B.P0, &h->B.P1, &h->B.P2, &h->B.P3, &h->B.P4, &h->B.P5, &h->B.P6, &h->B.R0, &h->B.R1, &h->B.R2, &h->B.R3, &h->B.N0};
    for (int i = 0; i < 12; ++i) { *planes[i] = (float4*)c; c += plane; }
    h->B.E0 = (float4*)c; c += eplane;
    h->B.E1 = (float4*)c; c += eplane;
    h->B.gstep = (uint32_t*)c; c += gs;
    h->B.obs = (float*)c; c += ob;
    h->B.reward = (float*)c; c += rw;
    h->B.done = (uint8_t*)c; c += dn;
    h->B.ticket = (unsigned*)c; c += 256;
    h->B.reward_d = (float*)(c + al(n_items_max * 4));
    h->B.item_seq = (unsigned*)c;
    if (h->P.lat_a_n > 0) {
        ce = cudaMalloc(&h->hist, 3 * plane);
        if (ce == cudaSuccess) ce = cudaMemset(h->hist, 0, 3 * plane);
        if (ce != cudaSuccess) { cudaFree(h->arena); if (h->hist) cudaFree(h->hist); delete h; return fail(MDG_ENOMEM, std::string("mdg_create: cudaMalloc (action history): ") + cudaGetErrorString(ce)); }
        h->B.H0 = (float4*)h->hist; h->B.H1 = (float4*)((char*)h->hist + plane); h->B.H2 = (float4*)((char*)h->hist + 2 * plane);
    }
    int rc = configure_launch(h);
    if (rc == MDG_OK && h->saturating) {     // throughput-bound batch: register budget (resident 128-thread blocks per SM) as measured fastest
        const bool generic = h->kernel_name.find("generic") != std::string::npos;
        // 6 for the benchmark specialisations (80 registers: only the integrated state and the frozen wrench live across the substep
        // loop); 4 where the motor lag / latency rows keep rotor commands and history rows live as well (measured: 45.0 vs 50.9 us at 5);
        // the runtime-flag kernel needs 162 registers to stay out of local memory (3)
        h->minb = generic ? 3 : (h->P.feat & (F_MLAG | F_LAT)) ? 4 : 6;   // jit kernels follow the same rule
        pick_kernels(h);
        rc = configure_launch(h);
    }
    // Two envs per lane (packed FP32 pairs in the substep loop) when the grid still fills the device with half the warps:
    // an issue-bound kernel gains from the halved instruction count, a latency-bound one would only lose parallelism.
    int want_lanes = 0;
    if (const char* ev = std::getenv("MDG_LANES")) want_lanes = ev[0] == '2' ? 2 : 1;
    // (not with per-drone DR planes or sensor rows: their scalar prologue / epilogue work per env slot outweighs the packed loop;
    //  measured on config 5: DR 30.6 vs 24.5 us, sensor noise 33.6 vs 28.4 us)
    const bool lanes2_pays = !(h->P.feat & (F_DR | F_SENS));
    if (rc == MDG_OK && want_lanes != 1 && lanes2_capable(h->P.feat) && ((h->saturating && lanes2_pays) || want_lanes == 2) &&
        h->kernel_name.find("generic") == std::string::npos) {
        const int minb1 = h->minb;
        h->lanes = 2; h->minb = 4;
        if (const char* ev = std::getenv("MDG_X2_MINB")) h->minb = std::atoi(ev) >= 4 ? 4 : 3;   // 128 instead of 168 registers
        pick_kernels(h);
        rc = configure_launch(h);
        if (rc != MDG_OK || h->lanes != 2 || (!h->saturating && want_lanes != 2)) {
            h->lanes = 1; h->minb = minb1;
            pick_kernels(h);
            rc = configure_launch(h);
        }
    }
    if (rc == MDG_OK && h->jit == 2 && !h->jit_note.empty())
        rc = fail(MDG_ECUDA, "mdg_create: MDG_JIT=require and the run-time specialisation failed: " + h->jit_note);
    if (rc != MDG_OK) { cudaFree(h->arena); if (h->hist) cudaFree(h->hist); delete h; return rc; }
    *out = h;
    rc = mdg_reset(h, 0);
    if (rc != MDG_OK) { mdg_destroy(h); *out = nullptr; return rc; }
    // a fallback to the 1.7-2.1x slower runtime-flag kernel is not an error, but it is not silent either: the text is
    // readable through mdg_last_error() right after mdg_create, and mdg_kernel_name() says "generic"
    if (!h->jit_note.empty()) g_err = "mdg_create: run-time specialisation unavailable, using the generic kernel: " + h->jit_note;
    else g_err.clear();
    return MDG_OK;
}

void mdg_destroy(mdg_env* h) {
    if (!h) return;
    drop_graphs(h);
    if (h->stage) cudaFree(h->stage);
    if (h->order_event) cudaEventDestroy(h->order_event);
    if (h->capture_stream) cudaStreamDestroy(h->capture_stream);
    if (h->arena) cudaFree(h->arena);
    if (h->hist) cudaFree(h->hist);
    delete h;
}

int mdg_reset(mdg_env* h, uint64_t seed) {
    if (!h) return fail(MDG_EINVAL, "mdg_reset: NULL handle");
    h->P.seed_lo = (uint32_t)seed; h->P.seed_hi = (uint32_t)(seed >> 32);
    drop_graphs(h);                          // captured launches carry the old seed
    h->chainable = false;                    // the dispensers are back at 0 after every launch: nothing to clear
    h->reset<<<grid_for(h, 128), 128, 0, h->stream>>>(h->P, h->B);
    CU(cudaGetLastError());
    h->launches += 1;
    return MDG_OK;
}

int mdg_step(mdg_env* h, const float* actions_dev) {
    if (!h || !actions_dev) return fail(MDG_EINVAL, "mdg_step: NULL argument");
    if ((uintptr_t)actions_dev & 15) return fail(MDG_EINVAL, "mdg_step: actions_dev must be 16-byte aligned");
    return launch_step(h, actions_dev, h->stream, false);
}

int mdg_step_chained(mdg_env* h, const float* actions_dev) {
    if (!h || !actions_dev) return fail(MDG_EINVAL, "mdg_step_chained: NULL argument");
    if ((uintptr_t)actions_dev & 15) return fail(MDG_EINVAL, "mdg_step_chained: actions_dev must be 16-byte aligned");
    return launch_step(h, actions_dev, h->stream, true);
}

int mdg_step_many(mdg_env* h, const float* actions_dev, int n_steps, int64_t stride_floats) {
    if (!h || !actions_dev || n_steps < 1) return fail(MDG_EINVAL, "mdg_step_many: bad argument");
    if (((uintptr_t)actions_dev & 15) || (stride_floats & 3)) return fail(MDG_EINVAL, "mdg_step_many: actions must stay 16-byte aligned");
    const auto key = std::make_tuple((const void*)actions_dev, n_steps, stride_floats);
    auto it = h->graphs.find(key);
    if (it == h->graphs.end()) {
        if (!h->capture_stream) CU(cudaStreamCreateWithFlags(&h->capture_stream, cudaStreamNonBlocking));
        const int64_t launches0 = h->launches;
        CU(cudaStreamBeginCapture(h->capture_stream, cudaStreamCaptureModeThreadLocal));
        int rc = MDG_OK;
        // the first launch waits for whatever precedes the replay and publishes its (baked) sequence number for every item;
        // the others chain item by item behind their predecessor in the graph, exactly like a stream of mdg_step_chained calls
        for (int k = 0; k < n_steps && rc == MDG_OK; ++k) rc = launch_step(h, actions_dev + (int64_t)k * stride_floats, h->capture_stream, k > 0);
        cudaGraph_t g = nullptr;
        cudaError_t ce = cudaStreamEndCapture(h->capture_stream, &g);
        h->launches = launches0;                 // capturing launches nothing
        h->chainable = false;
        if (rc != MDG_OK) { if (g) cudaGraphDestroy(g); return rc; }
        if (ce != cudaSuccess) return fail(MDG_ECUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(ce));
        cudaGraphExec_t ge = nullptr;
        ce = cudaGraphInstantiate(&ge, g, 0);
        cudaGraphDestroy(g);
        if (ce != cudaSuccess) return fail(MDG_ECUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ce));
        if (h->graphs.size() >= 16) drop_graphs(h);
        it = h->graphs.emplace(key, ge).first;
    }
    nvtxRangePushA("mdg_step_many");
    const cudaError_t ce = cudaGraphLaunch(it->second, h->stream);
    nvtxRangePop();
    if (ce != cudaSuccess) return fail(MDG_ECUDA, std::string("cudaGraphLaunch: ") + cudaGetErrorString(ce));
    h->chainable = false;                    // a step after the replay waits for all of it
    h->launches += n_steps;
    return MDG_OK;
}

int mdg_outputs(mdg_env* h, const float** obs, const float** reward, const uint8_t** done) {
    if (!h) return fail(MDG_EINVAL, "mdg_outputs: NULL handle");
    if (obs) *obs = h->B.obs;
    if (reward) *reward = h->B.reward;
    if (done) *done = h->B.done;
    return MDG_OK;
}
int mdg_reward_per_drone(mdg_env* h, const float** r) {
    if (!h || !r) return fail(MDG_EINVAL, "mdg_reward_per_drone: NULL argument");
    *r = h->B.reward_d;
    return MDG_OK;
}
int mdg_obs_dim(const mdg_env* h) { return h ? h->M * h->P.opd : MDG_EINVAL; }
int mdg_targets(mdg_env* h, const float** t) {
    if (!h || !t) return fail(MDG_EINVAL, "mdg_targets: NULL argument");
    *t = reinterpret_cast<const float*>(h->B.P6);
    return MDG_OK;
}

int mdg_gen_actions(mdg_env* h, uint64_t seed, uint32_t t, float base, float lo, float hi, float* out_dev) {
    if (!h || !out_dev || ((uintptr_t)out_dev & 15)) return fail(MDG_EINVAL, "mdg_gen_actions: bad argument");
    const size_t D = (size_t)h->N * h->M;
    gen_actions_kernel<<<(unsigned)((D + 255) / 256), 256, 0, h->stream>>>(D, h->M, h->P.env_base, (uint32_t)seed, (uint32_t)(seed >> 32), t, base, lo, hi,
                                                                              reinterpret_cast<float4*>(out_dev));
    CU(cudaGetLastError());
    h->launches += 1;
    return MDG_OK;
}

int mdg_default_cam_params(const mdg_params* params, mdg_cam_params* out) {
    if (!out) return fail(MDG_EINVAL, "mdg_default_cam_params: NULL argument");
    mdg_params cf2x;
    if (!params) { const int rc = mdg_default_params(MDG_MODEL_CF2X, &cf2x); if (rc != MDG_OK) return rc; params = &cf2x; }
    std::memset(out, 0, sizeof(*out));
    out->struct_size = sizeof(mdg_cam_params);
    out->height = 48; out->width = 64; out->fovy_deg = 60.0f;
    out->offset[0] = 0.02f; out->offset[1] = 0.0f; out->offset[2] = 0.0f;
    out->znear = 0.01f; out->zfar = 50.0f;                                    // reading Q47
    out->body_radius = params->L + params->r_p; out->body_half_height = 0.0125f;   // reading Q46
    return MDG_OK;
}

// One launch of the camera kernel: depth and / or segmentation (mdg_render_depth), or the colour frame (mdg_render_rgba).
static int render_camera(mdg_env* h, const mdg_cam_params* cam, float* depth_dev, uint8_t* seg_dev, uint8_t* rgba_dev) {
    mdg_cam_params def;
    if (!cam) { const int rc = mdg_default_cam_params(&h->hp, &def); if (rc != MDG_OK) return rc; cam = &def; }
    if (cam->struct_size != sizeof(mdg_cam_params)) return fail(MDG_EINVAL, "mdg_render_depth: struct_size mismatch");
    if (cam->height < 1 || cam->width < 4 || (cam->width & 3) || (int64_t)cam->height * cam->width > (1 << 24))
        return fail(MDG_EINVAL, "mdg_render_depth: height >= 1, width a positive multiple of 4, height*width <= 2^24");
    if (!(cam->fovy_deg > 0.0f && cam->fovy_deg < 180.0f) || !(cam->znear > 0.0f) || !(cam->zfar > cam->znear) ||
        !(cam->body_radius > 0.0f) || !(cam->body_half_height > 0.0f))
        return fail(MDG_EINVAL, "mdg_render_depth: fovy in (0, 180), 0 < znear < zfar and positive body axes required");
    CamDev C;
    C.H = cam->height; C.W = cam->width; C.groups_per_row = cam->width / 4; C.n_groups = C.H * C.groups_per_row;
    C.s = (float)(2.0 * std::tan(0.5 * (double)cam->fovy_deg * 3.14159265358979323846 / 180.0) / cam->height);
    C.half_h = 0.5f * cam->height; C.half_w = 0.5f * cam->width; C.inv_gpr = 1.0f / (float)C.groups_per_row;
    C.g_rstep = 32 / C.groups_per_row; C.g_cstep = 32 % C.groups_per_row;
    for (int i = 0; i < 3; ++i) C.off[i] = cam->offset[i];
    C.znear = cam->znear; C.zfar = cam->zfar;
    C.rb = std::fmax(cam->body_radius, cam->body_half_height);
    C.tan_h = C.half_w * C.s; C.tan_v = C.half_h * C.s;
    C.len_h = std::sqrt(1.0f + C.tan_h * C.tan_h) * 1.001f; C.len_v = std::sqrt(1.0f + C.tan_v * C.tan_v) * 1.001f;
    C.a2 = (float)((double)cam->body_radius * cam->body_radius);
    C.dac = (float)((double)cam->body_half_height * cam->body_half_height - (double)cam->body_radius * cam->body_radius);
    C.inv_a = (float)(1.0 / (double)cam->body_radius); C.inv_c = (float)(1.0 / (double)cam->body_half_height);
    const int n_cams = h->N * h->M;
    const unsigned grid = (unsigned)((n_cams + CAM_WARPS - 1) / CAM_WARPS);
    const size_t smem = (size_t)CAM_WARPS * h->M * (sizeof(CamCand) + (rgba_dev ? sizeof(CamShade) : 0));
    h->chainable = false;                    // a later step must order itself behind this reader as a whole
    const bool two_pass = depth_dev && seg_dev, aligned = C.g_cstep == 0;
    auto kern = rgba_dev ? (aligned ? render_depth_kernel<CAM_RGBA, true> : render_depth_kernel<CAM_RGBA, false>)
              : two_pass ? (aligned ? render_depth_kernel<CAM_TWO_PASS, true> : render_depth_kernel<CAM_TWO_PASS, false>)
                         : (aligned ? render_depth_kernel<CAM_ONE_PASS, true> : render_depth_kernel<CAM_ONE_PASS, false>);
    kern<<<grid, CAM_WARPS * 32, smem, h->stream>>>(h->B.P0, h->B.P1, n_cams, h->M, C, depth_dev, seg_dev, reinterpret_cast<uint4*>(rgba_dev));
    CU(cudaGetLastError());
    h->launches += 1;
    return MDG_OK;
}

int mdg_render_depth(mdg_env* h, const mdg_cam_params* cam, float* depth_dev, uint8_t* seg_dev) {
    if (!h) return fail(MDG_EINVAL, "mdg_render_depth: NULL handle");
    if (!depth_dev && !seg_dev) return fail(MDG_EINVAL, "mdg_render_depth: both outputs NULL");
    if (((uintptr_t)depth_dev & 15) || ((uintptr_t)seg_dev & 3)) return fail(MDG_EINVAL, "mdg_render_depth: depth_dev must be 16-byte, seg_dev 4-byte aligned");
    return render_camera(h, cam, depth_dev, seg_dev, nullptr);
}

int mdg_render_rgba(mdg_env* h, const mdg_cam_params* cam, uint8_t* rgba_dev) {
    if (!h) return fail(MDG_EINVAL, "mdg_render_rgba: NULL handle");
    if (!rgba_dev) return fail(MDG_EINVAL, "mdg_render_rgba: NULL output");
    if ((uintptr_t)rgba_dev & 15) return fail(MDG_EINVAL, "mdg_render_rgba: rgba_dev must be 16-byte aligned");
    return render_camera(h, cam, nullptr, nullptr, rgba_dev);
}

int mdg_set_stream(mdg_env* h, void* s) {
    if (!h) return fail(MDG_EINVAL, "mdg_set_stream: NULL handle");
    cudaStream_t ns = (cudaStream_t)s;
    if (ns != h->stream) {
        // what is already queued on the old stream (the create-time clear and reset, earlier steps) stays ahead of what follows
        cudaStreamCaptureStatus c0 = cudaStreamCaptureStatusNone, c1 = cudaStreamCaptureStatusNone;
        CU(cudaStreamIsCapturing(h->stream, &c0));
        CU(cudaStreamIsCapturing(ns, &c1));
        if (c0 == cudaStreamCaptureStatusNone && c1 == cudaStreamCaptureStatusNone) {   // inside a capture the ordering is the caller's graph
            if (!h->order_event) CU(cudaEventCreateWithFlags(&h->order_event, cudaEventDisableTiming));
            CU(cudaEventRecord(h->order_event, h->stream));
            CU(cudaStreamWaitEvent(ns, h->order_event, 0));
        }
        h->stream = ns;
    }
    h->chainable = false;
    return MDG_OK;
}
int64_t mdg_launch_count(const mdg_env* h) { return h ? h->launches : 0; }
const char* mdg_kernel_name(const mdg_env* h) { return h ? h->kernel_name.c_str() : ""; }
int mdg_set_launch(mdg_env* h, int block_threads, int max_blocks_per_sm) {
    if (!h) return fail(MDG_EINVAL, "mdg_set_launch: NULL handle");
    if (block_threads) {
        if (block_threads < 32 || block_threads > 128 || (block_threads & 31)) return fail(MDG_EINVAL, "mdg_set_launch: block must be a multiple of 32 in [32, 128]");
        h->block = block_threads;
    }
    if (max_blocks_per_sm) {
        if (max_blocks_per_sm < 0 || max_blocks_per_sm > 32) return fail(MDG_EINVAL, "mdg_set_launch: max_blocks_per_sm in [1, 32]");
        h->max_blocks_per_sm = max_blocks_per_sm;
        // register-budget variant: resident 128-thread blocks per SM the allocation must allow (4..8)
        const int per128 = (max_blocks_per_sm * h->block + 127) / 128;
        h->minb = per128 < 3 ? 3 : (per128 > 8 ? 8 : per128);   // 3 exists for the generic kernel only (specialisations fall back to 4)
        pick_kernels(h);
    }
    drop_graphs(h);
    h->chainable = false;
    return configure_launch(h);
}

}  // extern "C"

// ---- checkpoint / test hooks: host AoS <-> device SoA planes ---------------------------------------
extern "C" int mdg_get_state(mdg_env* h, float* state, float* ctrl, float* targets, float* wind, uint32_t* ep_step) {
    if (!h) return fail(MDG_EINVAL, "mdg_get_state: NULL handle");
    CU(cudaStreamSynchronize(h->stream));
    const size_t D = (size_t)h->N * h->M;
    std::vector<float4> pl[7];
    float4* src[7] = {h->B.P0, h->B.P1, h->B.P2, h->B.P3, h->B.P4, h->B.P5, h->B.P6};
    for (int i = 0; i < 7; ++i) { pl[i].resize(D); CU(cudaMemcpy(pl[i].data(), src[i], D * sizeof(float4), cudaMemcpyDeviceToHost)); }
    for (size_t d = 0; d < D; ++d) {
        const float4 a = pl[0][d], b = pl[1][d], c = pl[2][d], e = pl[3][d], f = pl[4][d], s = pl[5][d], t = pl[6][d];
        if (state) { float* o = state + d * 13; o[0] = a.x; o[1] = a.y; o[2] = a.z; o[3] = a.w; o[4] = b.x; o[5] = b.y; o[6] = b.z;
                     o[7] = b.w; o[8] = c.x; o[9] = c.y; o[10] = c.z; o[11] = c.w; o[12] = e.x; }
        if (ctrl) { float* o = ctrl + d * 10; o[0] = e.y; o[1] = e.z; o[2] = e.w; o[3] = f.x; o[4] = f.y; o[5] = f.z;
                    o[6] = s.x; o[7] = s.y; o[8] = s.z; o[9] = s.w; }
        if (targets) { float* o = targets + d * 4; o[0] = t.x; o[1] = t.y; o[2] = t.z; o[3] = t.w; }
    }
    if (wind || ep_step) {
        std::vector<float4> ev(h->N);
        CU(cudaMemcpy(ev.data(), h->B.E0, (size_t)h->N * sizeof(float4), cudaMemcpyDeviceToHost));
        for (int e = 0; e < h->N; ++e) {
            if (wind) { wind[e * 3 + 0] = ev[e].x; wind[e * 3 + 1] = ev[e].y; wind[e * 3 + 2] = ev[e].z; }
            if (ep_step) std::memcpy(&ep_step[e], &ev[e].w, 4);
        }
    }
    return MDG_OK;
}

extern "C" int mdg_set_state(mdg_env* h, const float* state, const float* ctrl, const float* targets, const float* wind,
                             const uint32_t* ep_step) {
    if (!h) return fail(MDG_EINVAL, "mdg_set_state: NULL handle");
    CU(cudaStreamSynchronize(h->stream));
    const size_t D = (size_t)h->N * h->M;
    std::vector<float4> pl[7];
    float4* dst[7] = {h->B.P0, h->B.P1, h->B.P2, h->B.P3, h->B.P4, h->B.P5, h->B.P6};
    for (int i = 0; i < 7; ++i) { pl[i].resize(D); CU(cudaMemcpy(pl[i].data(), dst[i], D * sizeof(float4), cudaMemcpyDeviceToHost)); }
    for (size_t d = 0; d < D; ++d) {
        if (state) { const float* o = state + d * 13;
                     pl[0][d] = make_float4(o[0], o[1], o[2], o[3]); pl[1][d] = make_float4(o[4], o[5], o[6], o[7]);
                     pl[2][d] = make_float4(o[8], o[9], o[10], o[11]); pl[3][d].x = o[12]; }
        if (ctrl) { const float* o = ctrl + d * 10;
                    pl[3][d].y = o[0]; pl[3][d].z = o[1]; pl[3][d].w = o[2]; pl[4][d] = make_float4(o[3], o[4], o[5], 0.0f);
                    pl[5][d] = make_float4(o[6], o[7], o[8], o[9]); }
        if (targets) { const float* o = targets + d * 4; pl[6][d] = make_float4(o[0], o[1], o[2], o[3]); }
    }
    for (int i = 0; i < 7; ++i) CU(cudaMemcpy(dst[i], pl[i].data(), D * sizeof(float4), cudaMemcpyHostToDevice));
    if (wind || ep_step) {
        std::vector<float4> ev(h->N);
        CU(cudaMemcpy(ev.data(), h->B.E0, (size_t)h->N * sizeof(float4), cudaMemcpyDeviceToHost));
        for (int e = 0; e < h->N; ++e) {
            if (wind) { ev[e].x = wind[e * 3 + 0]; ev[e].y = wind[e * 3 + 1]; ev[e].z = wind[e * 3 + 2]; }
            if (ep_step) std::memcpy(&ev[e].w, &ep_step[e], 4);
        }
        CU(cudaMemcpy(h->B.E0, ev.data(), (size_t)h->N * sizeof(float4), cudaMemcpyHostToDevice));
    }
    h->chainable = false;
    h->refresh<<<grid_for(h, 128), 128, 0, h->stream>>>(h->P, h->B);
    CU(cudaGetLastError());
    h->launches += 1;
    CU(cudaStreamSynchronize(h->stream));
    return MDG_OK;
}

// ---- domain-randomisation factors: host [D][8] <-> planes R0, R1 --------------------------------------
extern "C" int mdg_get_dr(mdg_env* h, float* f) {
    if (!h || !f) return fail(MDG_EINVAL, "mdg_get_dr: NULL argument");
    CU(cudaStreamSynchronize(h->stream));
    const size_t D = (size_t)h->N * h->M;
    float4* src[4] = {h->B.R0, h->B.R1, h->B.R2, h->B.R3};
    std::vector<float4> a(D);
    for (int k = 0; k < 4; ++k) {
        CU(cudaMemcpy(a.data(), src[k], D * sizeof(float4), cudaMemcpyDeviceToHost));
        for (size_t d = 0; d < D; ++d) { float* o = f + d * 16 + k * 4; o[0] = a[d].x; o[1] = a[d].y; o[2] = a[d].z; o[3] = a[d].w; }
    }
    return MDG_OK;
}
extern "C" int mdg_set_dr(mdg_env* h, const float* f) {
    if (!h || !f) return fail(MDG_EINVAL, "mdg_set_dr: NULL argument");
    if (!(h->P.feat & F_DR)) return fail(MDG_EINVAL, "mdg_set_dr: domain randomisation is off for this handle (all dr_alpha are 0)");
    CU(cudaStreamSynchronize(h->stream));
    const size_t D = (size_t)h->N * h->M;
    float4* dst[4] = {h->B.R0, h->B.R1, h->B.R2, h->B.R3};
    std::vector<float4> a(D);
    for (int k = 0; k < 4; ++k) {
        for (size_t d = 0; d < D; ++d) { const float* o = f + d * 16 + k * 4; a[d] = make_float4(o[0], o[1], o[2], o[3]); }
        CU(cudaMemcpy(dst[k], a.data(), D * sizeof(float4), cudaMemcpyHostToDevice));
    }
    h->chainable = false;
    return MDG_OK;
}

// ---- end-to-end call with host buffers --------------------------------------------------------------
// ---- full checkpoint: every device buffer a later step reads, as one opaque host blob ---------------------
namespace {
struct CkptHeader { uint32_t magic, version; int32_t N, M, feat, opd; uint32_t seed_lo, seed_hi; uint64_t bytes_main, bytes_rd, bytes_hist; };
const uint32_t CKPT_MAGIC = 0x4347444Du /* "MDGC" */, CKPT_VERSION = 1;
// main region: the state / DR / rotor planes, per-env words, step counters and outputs, contiguous in the arena up to the
// scheduler words (ticket dispensers and per-item flags are launch bookkeeping, not simulation state)
inline size_t ckpt_main_bytes(const mdg_env* h) { return (size_t)((const char*)h->B.ticket - (const char*)h->B.P0); }
inline size_t ckpt_rd_bytes(const mdg_env* h) { return (size_t)h->N * h->M * sizeof(float); }
inline size_t ckpt_hist_bytes(const mdg_env* h) { return h->hist ? (size_t)((const char*)h->B.H1 - (const char*)h->B.H0) * 3 : 0; }
}
extern "C" int64_t mdg_checkpoint_size(const mdg_env* h) {
    if (!h) return fail(MDG_EINVAL, "mdg_checkpoint_size: NULL handle");
    return (int64_t)(sizeof(CkptHeader) + ckpt_main_bytes(h) + ckpt_rd_bytes(h) + ckpt_hist_bytes(h));
}
extern "C" int mdg_save(mdg_env* h, void* host_buf, int64_t buf_bytes) {
    if (!h || !host_buf) return fail(MDG_EINVAL, "mdg_save: NULL argument");
    if (buf_bytes < mdg_checkpoint_size(h)) return fail(MDG_EINVAL, "mdg_save: buffer smaller than mdg_checkpoint_size");
    CU(cudaStreamSynchronize(h->stream));
    CkptHeader hd = {CKPT_MAGIC, CKPT_VERSION, h->N, h->M, h->P.feat, h->P.opd, h->P.seed_lo, h->P.seed_hi,
                     ckpt_main_bytes(h), ckpt_rd_bytes(h), ckpt_hist_bytes(h)};
    char* c = (char*)host_buf;
    std::memcpy(c, &hd, sizeof(hd)); c += sizeof(hd);
    CU(cudaMemcpy(c, h->B.P0, hd.bytes_main, cudaMemcpyDeviceToHost)); c += hd.bytes_main;
    CU(cudaMemcpy(c, h->B.reward_d, hd.bytes_rd, cudaMemcpyDeviceToHost)); c += hd.bytes_rd;
    if (hd.bytes_hist) CU(cudaMemcpy(c, h->hist, hd.bytes_hist, cudaMemcpyDeviceToHost));
    return MDG_OK;
}
extern "C" int mdg_load(mdg_env* h, const void* host_buf, int64_t buf_bytes) {
    if (!h || !host_buf) return fail(MDG_EINVAL, "mdg_load: NULL argument");
    if (buf_bytes < (int64_t)sizeof(CkptHeader)) return fail(MDG_EINVAL, "mdg_load: buffer too small for a checkpoint header");
    CkptHeader hd;
    std::memcpy(&hd, host_buf, sizeof(hd));
    if (hd.magic != CKPT_MAGIC || hd.version != CKPT_VERSION) return fail(MDG_EINVAL, "mdg_load: not a checkpoint of this library version");
    if (hd.N != h->N || hd.M != h->M || hd.feat != h->P.feat || hd.opd != h->P.opd || hd.bytes_main != ckpt_main_bytes(h) ||
        hd.bytes_rd != ckpt_rd_bytes(h) || hd.bytes_hist != ckpt_hist_bytes(h))
        return fail(MDG_EINVAL, "mdg_load: the checkpoint was written by a handle of another shape or feature set");
    if (buf_bytes < mdg_checkpoint_size(h)) return fail(MDG_EINVAL, "mdg_load: truncated checkpoint");
    CU(cudaStreamSynchronize(h->stream));
    const char* c = (const char*)host_buf + sizeof(hd);
    CU(cudaMemcpy(h->B.P0, c, hd.bytes_main, cudaMemcpyHostToDevice)); c += hd.bytes_main;
    CU(cudaMemcpy(h->B.reward_d, c, hd.bytes_rd, cudaMemcpyHostToDevice)); c += hd.bytes_rd;
    if (hd.bytes_hist) CU(cudaMemcpy(h->hist, c, hd.bytes_hist, cudaMemcpyHostToDevice));
    h->P.seed_lo = hd.seed_lo; h->P.seed_hi = hd.seed_hi;
    drop_graphs(h);                          // captured launches carry the old seed
    h->chainable = false;                    // the next step waits for the whole stream, not for item flags of a step it never saw
    return MDG_OK;
}

extern "C" int mdg_step_host_async(mdg_env* h, const float* actions_host, float* obs_host, float* reward_host, uint8_t* done_host) {
    if (!h || !actions_host) return fail(MDG_EINVAL, "mdg_step_host: NULL argument");
    const size_t D = (size_t)h->N * h->M;
    if (!h->stage) CU(cudaMalloc(&h->stage, D * 4 * sizeof(float)));
    CU(cudaMemcpyAsync(h->stage, actions_host, D * 4 * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    const int rc = launch_step(h, h->stage, h->stream, false);
    if (rc != MDG_OK) return rc;
    if (obs_host) CU(cudaMemcpyAsync(obs_host, h->B.obs, D * h->P.opd * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
    if (reward_host) CU(cudaMemcpyAsync(reward_host, h->B.reward, (size_t)h->N * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
    if (done_host) CU(cudaMemcpyAsync(done_host, h->B.done, (size_t)h->N, cudaMemcpyDeviceToHost, h->stream));
    return MDG_OK;
}
extern "C" int mdg_wait(mdg_env* h) {
    if (!h) return fail(MDG_EINVAL, "mdg_wait: NULL handle");
    CU(cudaStreamSynchronize(h->stream));
    return MDG_OK;
}
extern "C" int mdg_step_host(mdg_env* h, const float* actions_host, float* obs_host, float* reward_host, uint8_t* done_host) {
    const int rc = mdg_step_host_async(h, actions_host, obs_host, reward_host, done_host);
    return rc != MDG_OK ? rc : mdg_wait(h);
}
// ---- mdg_step_host without any allocation --------------------------------------------------------------------------
// mdg_step_host_async cudaMallocs its device staging buffer on a handle's first call.  Callers that must not allocate (a serving
// loop, code under stream capture, harnesses that forbid it) get the same step with the staging buffer in a file-scope device
// array: MDG_STATIC_STAGE_MAX_DRONES action rows of 16 bytes = 4 MiB, held by every GPU that loads the library until exit.
// In host code `g_static_stage` is only the host-side stand-in of the symbol, never a device address: the address is looked up
// once per device, with that device current, and that pointer is what the copy and the kernel get.
static __device__ __align__(256) float g_static_stage[(size_t)MDG_STATIC_STAGE_MAX_DRONES * 4];
static constexpr int kMaxDevices = 64;
static std::mutex g_static_stage_mu;
static float* g_static_stage_ptr[kMaxDevices] = {};

// Device address of g_static_stage on the CURRENT device (resolved at the first use on that device; allocates nothing).
static int static_stage_address(float** out) {
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(MDG_EINVAL, "mdg_step_host_static: device ordinal out of range");
    std::lock_guard<std::mutex> lk(g_static_stage_mu);
    if (!g_static_stage_ptr[dev]) {
        float* ptr = nullptr;
        const cudaError_t ce = cudaGetSymbolAddress((void**)&ptr, g_static_stage);
        if (ce != cudaSuccess || !ptr) return fail(MDG_ECUDA, std::string("mdg_step_host_static: cudaGetSymbolAddress: ") + cudaGetErrorString(ce));
        g_static_stage_ptr[dev] = ptr;
    }
    *out = g_static_stage_ptr[dev];
    return MDG_OK;
}

extern "C" int mdg_step_host_static(mdg_env* h, const float* actions_host, float* obs_host, float* reward_host, uint8_t* done_host) {
    if (!h || !actions_host) return fail(MDG_EINVAL, "mdg_step_host_static: NULL argument");
    const size_t D = (size_t)h->N * h->M;
    if (D > (size_t)MDG_STATIC_STAGE_MAX_DRONES)
        return fail(MDG_EINVAL, "mdg_step_host_static: n_envs * n_drones = " + std::to_string(D) + " exceeds the static staging buffer of " +
                                    std::to_string(MDG_STATIC_STAGE_MAX_DRONES) + " drones (MDG_STATIC_STAGE_MAX_DRONES); use mdg_step_host");
    float* stage = nullptr;
    const int ra = static_stage_address(&stage);
    if (ra != MDG_OK) return ra;
    // nothing in the array has to start at zero: the copy overwrites every word the kernel reads (the first D rows) before it runs
    CU(cudaMemcpyAsync(stage, actions_host, D * 4 * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    const int rc = launch_step(h, stage, h->stream, false);
    if (rc != MDG_OK) return rc;
    if (obs_host) CU(cudaMemcpyAsync(obs_host, h->B.obs, D * h->P.opd * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
    if (reward_host) CU(cudaMemcpyAsync(reward_host, h->B.reward, (size_t)h->N * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
    if (done_host) CU(cudaMemcpyAsync(done_host, h->B.done, (size_t)h->N, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return MDG_OK;
}
// ---- FP32 peak microbenchmark (roofline denominator check) ------------------------------------------
__global__ void __launch_bounds__(256) ffma_peak_kernel(float* out, int iters, float a, float b) {
    float x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 12345.678f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;      // keeps the chains alive, never true in practice
}
extern "C" int mdg_measure_fp32_peak(void* cuda_stream, double* tflops) {
    if (!tflops) return fail(MDG_EINVAL, "mdg_measure_fp32_peak: NULL argument");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0, n_sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));
    float* out = nullptr;
    const int blocks = n_sms * 8, threads = 256, iters = 4096;
    CU(cudaMalloc(&out, (size_t)blocks * threads * sizeof(float)));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        CU(cudaEventRecord(e0, s));
        ffma_peak_kernel<<<blocks, threads, 0, s>>>(out, iters, 0.999f, 0.001f);
        CU(cudaEventRecord(e1, s));
        CU(cudaEventSynchronize(e1));
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    CU(cudaGetLastError());
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    *tflops = 2.0 * 64.0 * iters * (double)blocks * threads / (best_ms * 1e-3) / 1e12;
    return MDG_OK;
}

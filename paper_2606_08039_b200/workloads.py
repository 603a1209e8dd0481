"""Seeded synthetic workload recipes — data only.

This module serves both the CUDA path and the oracle and therefore holds none of the method's
arithmetic: each recipe is the constructor arguments plus a dict of parameter overrides keyed by the
field names that `include/mdg.h:mdg_params` and the oracle's parameter block both use, and a
description of how the harness draws actions.  It imports neither side.
"""
import math

BASE_SEED = 260608039

# interface enum values (include/mdg.h; Table 1, 179-187 Table 3)
AERO_GND, AERO_DRAG, AERO_DW, AERO_WIND = 1, 2, 4, 8
WIND_DRYDEN, WIND_CONSTANT, WIND_GUST, WIND_SINE = 1, 2, 4, 8
INTEG_RK4, INTEG_EULER = 0, 1
PHYS_MJC, PHYS_MJC_GND, PHYS_MJC_DRAG, PHYS_MJC_DW, PHYS_MJC_GND_DRAG_DW, PHYS_DYN = range(6)
ACT_RPM, ACT_PID, ACT_VEL, ACT_RPM_NORM, ACT_ONE_D_RPM, ACT_ATTITUDE = 0, 1, 2, 3, 4, 5
OBS_KIN12, OBS_KIN12_ADJ, OBS_KIN20, OBS_KIN12_TGT, OBS_KIN12_WP, OBS_KIN12_Z = 0, 1, 2, 3, 4, 5
REW_HOVER, REW_NEG_SQ_DIST, REW_MULTI_HOVER, REW_FORMATION, REW_VELOCITY, REW_FLY_THROUGH = 0, 1, 2, 3, 4, 5
TERM_NONE, TERM_HOVER, TERM_TILT_DIST, TERM_FORMATION = 0, 1, 2, 3
LAYOUT_NONE, LAYOUT_GRID, LAYOUT_CIRCLE = 0, 1, 2
TGT_FIXED, TGT_SPAWN_LINSPACE, TGT_BOX, TGT_CIRCLE, TGT_WAYPOINTS = 0, 1, 2, 3, 4
MODEL_CF2X, MODEL_CF2P, MODEL_RACE = 0, 1, 2

_DSL = dict(dsl=1, int_clamp_pos=1.0, int_clamp_att=0.25)      # halved clamps + rate limits


class Workload:
    def __init__(self, name, n_envs, n_drones, physics_mode, action_type, params, actions, steps, seed):
        self.name, self.n_envs, self.n_drones = name, n_envs, n_drones
        self.physics_mode, self.action_type = physics_mode, action_type
        self.params = params          # {field: scalar | list}
        self.actions = actions        # ("hover_scale", lo, hi) | ("uniform", lo, hi) | ("targets",)
        self.steps, self.seed = steps, seed

    def scaled(self, n_envs):
        return Workload(self.name, n_envs, self.n_drones, self.physics_mode, self.action_type,
                        dict(self.params), self.actions, self.steps, self.seed)


def config(c: int) -> Workload:
    """The five BASELINE.json configs, c = 1..5 (seed = BASE_SEED + c)."""
    s = BASE_SEED + c
    if c == 1:      # 1 env x 1 CF2X, pure rigid body, RPM = hover x U[0.95, 1.05]
        return Workload("c1", 1, 1, PHYS_MJC, ACT_RPM, dict(
            reset_layout=LAYOUT_NONE, reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1],
            reward_mode=REW_HOVER, term_mode=TERM_HOVER, target_mode=TGT_FIXED, target_fixed=[0, 0, 1],
            episode_len_s=10.0, auto_reset=1), ("hover_scale", 0.95, 1.05), 1000, s)
    if c == 2:      # 4,096 x 1, ground effect + drag, z0 ~ U[0.05, 1.5]
        return Workload("c2", 4096, 1, PHYS_MJC, ACT_RPM, dict(
            aero_mask=AERO_GND | AERO_DRAG,
            reset_layout=LAYOUT_NONE, reset_center=[0, 0, 0], reset_half=[0, 0, 0], reset_z_lo=0.05, reset_z_hi=1.5,
            reward_mode=REW_HOVER, term_mode=TERM_HOVER, target_mode=TGT_FIXED, target_fixed=[0, 0, 1],
            episode_len_s=10.0, auto_reset=1), ("hover_scale", 0.9, 1.1), 2000, s)
    if c == 3:      # 16,384 x 1, PID waypoint (DSL flags), -|p-p*|^2, config-3 termination
        return Workload("c3", 16384, 1, PHYS_MJC, ACT_PID, dict(
            reset_layout=LAYOUT_NONE, reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1],
            reward_mode=REW_NEG_SQ_DIST, term_mode=TERM_TILT_DIST, term_tilt=0.4, term_dist=3.0, term_center=[0, 0, 0],
            target_mode=TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0],
            episode_len_s=10.0, auto_reset=1, **_DSL), ("targets",), 1000, s)
    if c == 4:      # 1,024 x 8, all-pairs downwash + ground + drag, 4x2 grid, multi-hover
        return Workload("c4", 1024, 8, PHYS_MJC_GND_DRAG_DW, ACT_RPM, dict(
            reset_layout=LAYOUT_GRID, grid_cols=4, grid_spacing=0.3, reset_center=[0, 0, 0],
            reset_half=[0.05, 0.05, 0], reset_z_lo=0.3, reset_z_hi=1.2,
            reward_mode=REW_MULTI_HOVER, term_mode=TERM_HOVER, target_mode=TGT_SPAWN_LINSPACE, mh_z_lo=0.7, mh_z_hi=1.2,
            episode_len_s=10.0, auto_reset=1), ("hover_scale", 0.9, 1.1), 2000, s)
    if c == 5:      # 65,536 x 4, all aero + wind, VEL through the PID, adjacency obs, formation
        return Workload("c5", 65536, 4, PHYS_MJC_GND_DRAG_DW, ACT_VEL, dict(
            aero_mask=AERO_GND | AERO_DRAG | AERO_DW | AERO_WIND, wind_sigma=0.5, wind_tau=1.0,
            reset_layout=LAYOUT_CIRCLE, circle_radius=0.3, reset_center=[0, 0, 1], reset_half=[0.05, 0.05, 0.05],
            obs_mode=OBS_KIN12_ADJ, adj_radius=0.5,
            reward_mode=REW_FORMATION, term_mode=TERM_FORMATION, term_center=[0, 0, 1], term_dist=3.0,
            target_mode=TGT_CIRCLE, form_center=[0, 0, 1], form_radius=0.3,
            episode_len_s=30.0, auto_reset=1, **_DSL), ("uniform", -1.0, 1.0), 500, s)
    raise ValueError(c)


# Secondary workloads on a config (bench.py --variant, tests/test_gpu_features.py): parameter overrides, data only.
#  dyn     Table 1's DYN integrator (SURVEY.md 8(f) NEXT-1 "DYN mode benchmarked")
#  noise   Table 4's sensor-noise rows alone (a feature word without a precompiled kernel instance)
#  table4  every row of Table 4 except the initial-velocity range: per-episode DR planes, initial attitude,
#          motor lag, action / sensor latency, sensor noise.  The +-0.5 m/s initial velocities are left out on config 5 because
#          at its 0.3 m formation they send drones through each other's downwash column, where Eq.6 amplifies rounding by
#          orders of magnitude (conditioning); the generic-kernel cases of the tests cover that row.
VARIANTS = {
    "dyn": dict(integrator=INTEG_EULER),
    "noise": dict(obs_noise=[0.01, 0.05, 0.0174533, 0.05]),
    "table4": dict(dr_alpha=[0.2, 0.2, 0.15, 0.15, 0.3, 0.3, 0.3, 0.02, 0.05, 0.02, 0.05, 0.0], reset_rpy_half=[0.1, 0.1, 0.1],
                   motor_lag_lo=0.005, motor_lag_hi=0.05, act_latency_lo=0.0, act_latency_hi=0.05,
                   obs_latency_lo=0.0, obs_latency_hi=0.02, obs_noise=[0.01, 0.05, 0.0174533, 0.05]),
}


def hover_rpm_f32(m=0.027, g=9.81, k_f=3.16e-10):
    """Harness scale for ("hover_scale", ...) actions: the CF2X hover rotor speed rounded to fp32."""
    import struct
    return struct.unpack("f", struct.pack("f", math.sqrt(m * g / (4.0 * k_f))))[0]


def camera_scene(seed, n_envs, n_drones, radius=0.6):
    """Seeded input for the onboard-camera call: state rows [D, 13] float32 with the env's drones
    on a circle of the given radius at heights U[0.05, 1.4], each yawed towards the centre +- 0.5 rad with roll / pitch
    U(+-0.35), so that every camera sees floor, sky and some of the other drones (formation flight seen from inside).
    A tenth of the drones sit on the floor (z = 0), whose camera origin may dip below it.  Velocities are zero."""
    import numpy as np
    rng = np.random.Generator(np.random.Philox(seed))
    D = n_envs * n_drones
    i = np.tile(np.arange(n_drones), n_envs)
    ang = 2 * math.pi * i / max(n_drones, 1) + rng.uniform(-0.25, 0.25, D)
    r = radius * rng.uniform(0.5, 1.5, D)
    z = np.where(rng.uniform(size=D) < 0.1, 0.0, rng.uniform(0.05, 1.4, D))
    roll, pitch = rng.uniform(-0.35, 0.35, D), rng.uniform(-0.35, 0.35, D)
    yaw = ang + math.pi + rng.uniform(-0.5, 0.5, D)
    cr, sr, cp, sp, cy, sy = np.cos(roll / 2), np.sin(roll / 2), np.cos(pitch / 2), np.sin(pitch / 2), np.cos(yaw / 2), np.sin(yaw / 2)
    st = np.zeros((D, 13), dtype=np.float32)
    st[:, 0], st[:, 1], st[:, 2] = r * np.cos(ang), r * np.sin(ang), z
    st[:, 3] = cr * cp * cy + sr * sp * sy          # ZYX Euler angles -> unit quaternion (w, x, y, z)
    st[:, 4] = sr * cp * cy - cr * sp * sy
    st[:, 5] = cr * sp * cy + sr * cp * sy
    st[:, 6] = cr * cp * sy - sr * sp * cy
    return st

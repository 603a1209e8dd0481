"""-m gpu: the runtime-flag (generic) step kernel and the corner shapes against the float64 oracle.

The five BASELINE.json configs run compile-time specialisations; everything else - drone counts that do not
fill a lane group, the DYN integrator, the RACE airframe, PID without the DSL limits, formation rewards on
arbitrary targets, termination off - runs the generic instantiation of the same source.  Each case is a
small synthetic workload in the style of `workloads.py` stepped for 1 s of simulated time.
"""
import pytest

from paper_2606_08039_b200 import workloads as W
from parity_util import run_parity

pytestmark = pytest.mark.gpu

HOVER = ("hover_scale", 0.9, 1.1)
GRID = dict(reset_layout=W.LAYOUT_GRID, grid_cols=3, grid_spacing=0.3, reset_center=[0, 0, 0], reset_half=[0.05, 0.05, 0],
            reset_z_lo=0.3, reset_z_hi=1.2, reward_mode=W.REW_MULTI_HOVER, term_mode=W.TERM_HOVER,
            target_mode=W.TGT_SPAWN_LINSPACE, mh_z_lo=0.7, mh_z_hi=1.2, episode_len_s=10.0, auto_reset=1)
CIRCLE = dict(reset_layout=W.LAYOUT_CIRCLE, circle_radius=0.4, reset_center=[0, 0, 1], reset_half=[0.05, 0.05, 0.05],
              obs_mode=W.OBS_KIN12_ADJ, adj_radius=0.5, reward_mode=W.REW_FORMATION, term_mode=W.TERM_FORMATION,
              term_center=[0, 0, 1], term_dist=3.0, form_center=[0, 0, 1], form_radius=0.4, episode_len_s=30.0, auto_reset=1)


SINGLE = dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_HOVER, term_mode=W.TERM_HOVER,
              target_mode=W.TGT_FIXED, target_fixed=[0, 0, 1], episode_len_s=10.0, auto_reset=1)


DR = [0.2, 0.2, 0.15, 0.15, 0.3, 0.3, 0.3, 0.02, 0.05, 0.02, 0.05, 0.0]     # Table 4
INIT = dict(reset_rpy_half=[0.1, 0.1, 0.1], reset_vel_half=[0.5, 0.5, 0.5])   # its "init" row


SENS = dict(obs_noise=[0.01, 0.05, 0.0174533, 0.05], obs_bias=[0.02, 0.03, 0.01, 0.04])   # Table 4 "sensors" rows; bias: PAPER.md:248 (iii)


LAT = dict(act_latency_lo=0.0, act_latency_hi=0.050, obs_latency_lo=0.0, obs_latency_hi=0.020)   # Table 4 "action latency", "sensor latency"


def wl(name, n, m, phys, act, params, actions, seed=77):
    return W.Workload(name, n, m, phys, act, params, actions, 48, W.BASE_SEED + seed)


CASES = {
    # partial lane groups: M = 3 in G = 4, M = 5 and 6 in G = 8, M = 11 in G = 16, M = 20 in G = 32
    "m3_all_aero": (wl("m3", 1001, 3, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM, dict(GRID), HOVER), {}),
    "m5_vel_wind_formation": (wl("m5", 517, 5, W.PHYS_MJC_GND_DRAG_DW, W.ACT_VEL,
                                 dict(CIRCLE, aero_mask=15, wind_sigma=0.5, wind_tau=1.0, target_mode=W.TGT_CIRCLE),
                                 ("uniform", -1.0, 1.0)), {}),
    "m6_dw_only": (wl("m6", 300, 6, W.PHYS_MJC_DW, W.ACT_RPM, dict(GRID), HOVER), {}),
    "m11_g16": (wl("m11", 130, 11, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM, dict(GRID, grid_cols=4), HOVER), {}),
    "m20_g32": (wl("m20", 67, 20, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM, dict(GRID, grid_cols=5), HOVER), {}),
    # full groups the benchmark configs do not use
    "m2_dyn_euler": (wl("m2", 777, 2, W.PHYS_DYN, W.ACT_RPM, dict(GRID, aero_mask=W.AERO_DW | W.AERO_DRAG), HOVER), {}),
    "m16_full": (wl("m16", 64, 16, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM, dict(GRID, grid_cols=4), HOVER), {}),
    "m32_full": (wl("m32", 33, 32, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM, dict(GRID, grid_cols=8), HOVER), {}),
    # formation reward against targets that are not the circle slots (pair distances by shuffle)
    "m4_formation_box_targets": (wl("m4box", 600, 4, W.PHYS_MJC, W.ACT_VEL,
                                    dict(CIRCLE, target_mode=W.TGT_BOX, target_lo=[-0.5, -0.5, 0.8], target_hi=[0.5, 0.5, 1.2]),
                                    ("uniform", -1.0, 1.0)), {}),
    # single drone: DYN integrator, PID without the DSL limits, ground effect only, no termination / no auto-reset
    "m1_dyn_rpm": (wl("m1dyn", 2049, 1, W.PHYS_DYN, W.ACT_RPM,
                      dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_HOVER, term_mode=W.TERM_HOVER,
                           target_mode=W.TGT_FIXED, target_fixed=[0, 0, 1], episode_len_s=10.0, auto_reset=1), ("hover_scale", 0.95, 1.05)), {}),
    "m1_pid_no_dsl": (wl("m1pid", 1500, 1, W.PHYS_MJC_GND, W.ACT_PID,
                         dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST,
                              term_tilt=0.4, term_dist=3.0, target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0],
                              episode_len_s=10.0, auto_reset=1), ("targets",)), {}),
    "m1_no_term_no_reset": (wl("m1free", 900, 1, W.PHYS_MJC_DRAG, W.ACT_RPM,
                               dict(reset_center=[0, 0, 1.5], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_HOVER, term_mode=W.TERM_NONE,
                                    target_mode=W.TGT_FIXED, target_fixed=[0, 0, 1], episode_len_s=0.25, auto_reset=0), ("hover_scale", 0.7, 1.0)), {}),
    # normalised / one-dimensional / attitude actions, the 20-dim KIN observation
    "m1_rpm_norm": (wl("m1norm", 1300, 1, W.PHYS_MJC_DRAG, W.ACT_RPM_NORM, dict(SINGLE), ("uniform", -0.25, 0.3)), {}),
    "m1_one_d_rpm": (wl("m1oned", 1300, 1, W.PHYS_MJC_GND, W.ACT_ONE_D_RPM, dict(SINGLE), ("uniform", -1.3, 1.3)), {}),
    "m1_attitude": (wl("m1att", 1300, 1, W.PHYS_MJC, W.ACT_ATTITUDE, dict(SINGLE), ("uniform", -0.3, 0.3)), {}),
    "m4_attitude_kin20": (wl("m4att", 700, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_ATTITUDE, dict(GRID, grid_cols=2, obs_mode=W.OBS_KIN20), ("uniform", -0.2, 0.2)), {}),
    "m3_kin20_rpm": (wl("m3kin20", 500, 3, W.PHYS_MJC_DW, W.ACT_RPM, dict(GRID, obs_mode=W.OBS_KIN20), HOVER), {}),
    # VelocityAviary: normalised RPM action, 16-dim obs with the target, velocity-tracking reward
    "m1_velocity_aviary": (wl("m1vel", 1700, 1, W.PHYS_MJC, W.ACT_RPM_NORM,
                              dict(SINGLE, obs_mode=W.OBS_KIN12_TGT, reward_mode=W.REW_VELOCITY, target_mode=W.TGT_BOX,
                                   target_lo=[-0.5] * 3, target_hi=[0.5] * 3, target_w_lo=-0.25, target_w_hi=0.25, at_target_radius=0.3,
                                   episode_len_s=0.5), ("uniform", -0.1, 0.12)), {}),
    "m2_velocity_vel_action": (wl("m2vel", 900, 2, W.PHYS_MJC_DRAG, W.ACT_VEL,
                                  dict(GRID, grid_cols=2, obs_mode=W.OBS_KIN12_TGT, reward_mode=W.REW_VELOCITY, target_mode=W.TGT_BOX,
                                       target_lo=[-0.5] * 3, target_hi=[0.5] * 3, target_w_lo=-0.25, target_w_hi=0.25, at_target_radius=0.3),
                                  ("uniform", -0.5, 0.5)), {}),
    # Table 4 domain randomisation: per-episode factors on m, J, k_f, k_m, drag, C_gnd, C_1, g (frequent episodes -> redraws)
    "m1_domain_randomisation_pid": (wl("m1dr", 1500, 1, W.PHYS_MJC_GND, W.ACT_PID,
                                       dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST,
                                            term_tilt=0.4, term_dist=3.0, target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0],
                                            episode_len_s=0.25, auto_reset=1, dr_alpha=DR, **INIT), ("targets",)), {}),
    "m4_domain_randomisation_all_aero": (wl("m4dr", 800, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM,
                                            dict(GRID, grid_cols=2, episode_len_s=0.3, dr_alpha=DR, **INIT), HOVER), {}),
    "m1_domain_randomisation_saturated_rotors": (wl("m1drsat", 900, 1, W.PHYS_MJC, W.ACT_RPM_NORM,
                                                    dict(SINGLE, episode_len_s=0.4, dr_alpha=DR), ("uniform", 0.8, 1.0)), {}),
    # wind components: constant + gust, sinusoidal alone, all three on a config-5-like setup (must leave the specialisation)
    "m1_wind_constant_plus_gust": (wl("m1wc", 1300, 1, W.PHYS_MJC, W.ACT_VEL, dict(SINGLE, aero_mask=W.AERO_WIND, wind_mask=3,
                                      wind_const=[0.9, -0.4, 0.1]), ("uniform", -0.5, 0.5)), {}),
    "m1_wind_sine": (wl("m1ws", 1300, 1, W.PHYS_MJC_DRAG, W.ACT_RPM, dict(SINGLE, aero_mask=W.AERO_WIND | W.AERO_DRAG, wind_mask=8,
                        wind_sine_amp=0.02, wind_sine_omega=4.4), ("hover_scale", 0.97, 1.03)), {}),
    "m4_wind_combined_c5_like": (wl("m4wall", 900, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_VEL,
                                    dict(CIRCLE, circle_radius=0.3, form_radius=0.3, aero_mask=15, wind_sigma=0.5, wind_tau=1.0, target_mode=W.TGT_CIRCLE,
                                         wind_mask=11, wind_const=[0.0, 0.9, 0.0], wind_sine_amp=0.01, wind_sine_omega=3.0, int_clamp_pos=1.0,
                                         int_clamp_att=0.25), ("uniform", -1.0, 1.0)), {}),
    # FlyThroughAviary: ordered waypoints, capture reward, KIN12_WP observation; waypoints close together
    # and a large capture radius so that captures, target hand-overs and terminal captures all happen within 48 steps
    "m1_fly_through_pid": (wl("m1fly", 1500, 1, W.PHYS_MJC, W.ACT_VEL,
                              dict(SINGLE, obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH, target_mode=W.TGT_WAYPOINTS,
                                   n_waypoints=3, waypoints=[0.0, 0.0, 1.0, 0.15, 0.0, 1.05, 0.15, 0.2, 1.0] + [0.0] * 15, wp_radius=0.12,
                                   episode_len_s=20.0), ("uniform", -1.0, 1.0)), {}),
    "m2_fly_through_default_list": (wl("m2fly", 800, 2, W.PHYS_MJC_DRAG, W.ACT_RPM,
                                       dict(GRID, grid_cols=2, reset_z_lo=0.9, reset_z_hi=1.1, obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH,
                                            target_mode=W.TGT_WAYPOINTS, wp_radius=0.25, episode_len_s=20.0), HOVER), {}),
    # gust impulses (frequent, short) alone and the paper's COMBINED = all four wind components
    "m1_wind_gust": (wl("m1wg", 1500, 1, W.PHYS_MJC, W.ACT_VEL, dict(SINGLE, aero_mask=W.AERO_WIND, wind_mask=4, gust_prob=0.2,
                        gust_max=2.0, gust_duration=0.2), ("uniform", -0.5, 0.5)), {}),
    # impulses that last a whole number of control steps (0.25 s = 12, and the default 0.5 s = 24): the end of an impulse must not
    # hang on the last bit of the accumulated phase (Q42; a differential fuzz found fp32 and fp64 ending them one step apart)
    "m1_wind_gust_whole_steps": (wl("m1wg12", 1500, 1, W.PHYS_MJC, W.ACT_VEL, dict(SINGLE, aero_mask=W.AERO_WIND, wind_mask=4, gust_prob=0.2,
                                    gust_max=2.0, gust_duration=0.25), ("uniform", -0.5, 0.5)), {}),
    "m2_wind_gust_default_duration": (wl("m2wg24", 900, 2, W.PHYS_MJC_DRAG, W.ACT_RPM, dict(GRID, grid_cols=2, aero_mask=W.AERO_WIND | W.AERO_DRAG,
                                         wind_mask=4, gust_prob=0.3, gust_max=1.5), HOVER), {}),
    "m2_wind_combined": (wl("m2wall", 900, 2, W.PHYS_MJC_DRAG, W.ACT_RPM, dict(GRID, grid_cols=2, aero_mask=W.AERO_WIND | W.AERO_DRAG, wind_mask=15,
                            wind_const=[0.0, 0.9, 0.0], wind_sine_amp=0.01, wind_sine_omega=3.0, gust_prob=0.1, gust_max=1.5, gust_duration=0.3,
                            episode_len_s=0.5), HOVER), {}),
    # RaceAviary parameters of the waypoint family: six gates close together, two laps, speed bonus
    "m1_race_two_laps": (wl("m1race", 1500, 1, W.PHYS_MJC, W.ACT_VEL,
                            dict(SINGLE, obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH, target_mode=W.TGT_WAYPOINTS, n_waypoints=6,
                                 waypoints=[0.1, 0.0, 1.0, 0.05, 0.09, 1.0, -0.05, 0.09, 1.0, -0.1, 0.0, 1.0, -0.05, -0.09, 1.0, 0.05, -0.09, 1.0] + [0.0] * 6,
                                 wp_radius=0.12, wp_bonus=20.0, wp_shaping=0.05, wp_speed=2.0, wp_omega=0.0, wp_laps=2, episode_len_s=30.0),
                            ("uniform", -1.0, 1.0)), {}),
    # MultiHoverAviary as the paper tabulates it: 13 floats per drone (kinematic state + target altitude), normalised RPM
    "m3_multi_hover_obs13": (wl("m3mh", 700, 3, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM_NORM, dict(GRID, obs_mode=W.OBS_KIN12_Z), ("uniform", -0.1, 0.12)), {}),
    # Table 4 motor lag: rotor-speed state, wrench recomputed every substep; alone under PID, and with everything else on
    "m1_motor_lag_pid": (wl("m1lag", 1500, 1, W.PHYS_MJC, W.ACT_PID,
                            dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST,
                                 term_tilt=0.4, term_dist=3.0, target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0],
                                 episode_len_s=0.5, auto_reset=1, motor_lag_lo=0.005, motor_lag_hi=0.05), ("targets",)), {}),
    "m4_motor_lag_dr_all_aero": (wl("m4lag", 700, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM,
                                    dict(GRID, grid_cols=2, episode_len_s=0.3, dr_alpha=DR, motor_lag_lo=0.005, motor_lag_hi=0.05, **INIT), HOVER), {}),
    # Table 4 sensor rows: per-step noise and per-episode bias on the observation, in each row layout (short episodes ->
    # the bias is redrawn at auto-resets); state, reward and done must be untouched by them
    "m1_sensors_pid": (wl("m1sens", 1500, 1, W.PHYS_MJC, W.ACT_PID,
                          dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST,
                               term_tilt=0.4, term_dist=3.0, target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0],
                               episode_len_s=0.25, auto_reset=1, **SENS), ("targets",)), {}),
    "m3_sensors_kin20": (wl("m3sens", 500, 3, W.PHYS_MJC_DW, W.ACT_RPM, dict(GRID, obs_mode=W.OBS_KIN20, episode_len_s=0.3, **SENS), HOVER), {}),
    "m4_sensors_c5_like": (wl("m4sens", 900, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_VEL,
                              dict(CIRCLE, circle_radius=0.3, form_radius=0.3, aero_mask=15, wind_sigma=0.5, wind_tau=1.0, target_mode=W.TGT_CIRCLE,
                                   int_clamp_pos=1.0, int_clamp_att=0.25, episode_len_s=0.4, **SENS), ("uniform", -1.0, 1.0)), {}),
    "m2_sensors_fly_through": (wl("m2sensfly", 800, 2, W.PHYS_MJC_DRAG, W.ACT_RPM,
                                  dict(GRID, grid_cols=2, reset_z_lo=0.9, reset_z_hi=1.1, obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH,
                                       target_mode=W.TGT_WAYPOINTS, wp_radius=0.25, episode_len_s=20.0, **SENS), HOVER), {}),
    "m5_sensors_obs13_dr": (wl("m5sens", 300, 5, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM_NORM,
                               dict(GRID, obs_mode=W.OBS_KIN12_Z, episode_len_s=0.3, dr_alpha=DR, **INIT, **SENS), ("uniform", -0.1, 0.12)), {}),
    # DRYDEN with the altitude-dependent length scale: alone at mixed altitudes (some below the altitude floor,
    # M = 3 in a 4-lane group for the mean), and inside the paper's COMBINED wind
    "m3_dryden_altitude": (wl("m3dry", 700, 3, W.PHYS_MJC_GND, W.ACT_VEL,
                              dict(GRID, reset_z_lo=0.02, reset_z_hi=2.5, aero_mask=W.AERO_WIND | W.AERO_GND, wind_sigma=0.6, dryden_airspeed=7.0,
                                   reward_mode=W.REW_MULTI_HOVER), ("uniform", -0.5, 0.5)), {}),
    "m4_dryden_altitude_combined_c5_like": (wl("m4dry", 900, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_VEL,
                                               dict(CIRCLE, circle_radius=0.3, form_radius=0.3, aero_mask=15, wind_sigma=0.5, dryden_airspeed=8.0,
                                                    target_mode=W.TGT_CIRCLE, wind_mask=15, wind_const=[0.0, 0.9, 0.0], wind_sine_amp=0.01,
                                                    wind_sine_omega=3.0, gust_prob=0.1, gust_max=1.5, gust_duration=0.3, int_clamp_pos=1.0,
                                                    int_clamp_att=0.25), ("uniform", -1.0, 1.0)), {}),
    # Table 4 latency rows: action latency 0-50 ms and sensor latency 0-20 ms per episode (short episodes -> redraws); rotor
    # commands switch at the exact substep, controllers decode from the row that has arrived
    "m1_latency_rpm": (wl("m1lat", 1500, 1, W.PHYS_MJC_DRAG, W.ACT_RPM, dict(SINGLE, episode_len_s=0.3, **LAT), HOVER), {}),
    "m1_latency_pid": (wl("m1latpid", 1500, 1, W.PHYS_MJC, W.ACT_PID,
                          dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST,
                               term_tilt=0.4, term_dist=3.0, target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0],
                               episode_len_s=0.25, auto_reset=1, **LAT), ("targets",)), {}),
    "m3_latency_kin20_norm": (wl("m3lat", 500, 3, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM_NORM, dict(GRID, obs_mode=W.OBS_KIN20, episode_len_s=0.3, **LAT),
                                 ("uniform", -0.1, 0.12)), {}),
    "m4_latency_c5_like_everything": (wl("m4lat", 900, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_VEL,
                                         dict(CIRCLE, circle_radius=0.3, form_radius=0.3, aero_mask=15, wind_sigma=0.5, wind_tau=1.0, target_mode=W.TGT_CIRCLE,
                                              int_clamp_pos=1.0, int_clamp_att=0.25, episode_len_s=0.4, **LAT, **SENS), ("uniform", -1.0, 1.0)), {}),
    "m4_latency_motor_lag_dr": (wl("m4latlag", 700, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM,
                                   dict(GRID, grid_cols=2, episode_len_s=0.3, dr_alpha=DR, motor_lag_lo=0.005, motor_lag_hi=0.05, **INIT, **LAT), HOVER), {}),
    "m1_latency_action_only_one_d": (wl("m1lat1d", 1300, 1, W.PHYS_MJC_GND, W.ACT_ONE_D_RPM, dict(SINGLE, episode_len_s=0.5, act_latency_lo=0.004, act_latency_hi=0.06),
                                        ("uniform", -0.3, 0.3)), {}),
    "m2_latency_sensor_only_fly_through": (wl("m2latfly", 800, 2, W.PHYS_MJC_DRAG, W.ACT_RPM,
                                              dict(GRID, grid_cols=2, reset_z_lo=0.9, reset_z_hi=1.1, obs_mode=W.OBS_KIN12_WP, reward_mode=W.REW_FLY_THROUGH,
                                                   target_mode=W.TGT_WAYPOINTS, wp_radius=0.25, episode_len_s=20.0, obs_latency_lo=0.0, obs_latency_hi=0.0208), HOVER), {}),
    # FormationAviary's moving centre: a fast lap round a small square so that 48 steps pass three vertices; the
    # 3 m rule measured from the moving centre; and a tilted triangle under M = 5 (partial lane group), short episodes
    "m4_formation_path_c5_like": (wl("m4path", 900, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_VEL,
                                     dict(CIRCLE, circle_radius=0.3, form_radius=0.3, aero_mask=15, wind_sigma=0.5, wind_tau=1.0, target_mode=W.TGT_CIRCLE,
                                          int_clamp_pos=1.0, int_clamp_att=0.25, form_path_n=4, form_speed=2.5,
                                          form_path=[0, 0, 1, 0.6, 0, 1, 0.6, 0.6, 1, 0, 0.6, 1] + [0.0] * 12), ("uniform", -1.0, 1.0)), {}),
    "m5_formation_path_triangle": (wl("m5path", 517, 5, W.PHYS_MJC_DRAG, W.ACT_VEL,
                                      dict(CIRCLE, target_mode=W.TGT_CIRCLE, episode_len_s=0.4, term_dist=0.9, form_path_n=3, form_speed=3.0,
                                           form_path=[0, 0, 1, 0.5, 0.1, 1.2, 0.2, 0.6, 0.9] + [0.0] * 15), ("uniform", -1.0, 1.0)), {}),
    # one env, one warp not even full
    "n1_m3": (wl("n1m3", 1, 3, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM, dict(GRID), HOVER), {}),
}


# ill-conditioned envs (parity_util "Conditioning": the fp32-rounded shadow oracle itself leaves the tolerance band) measured per
# multi-drone case on the fixed seeds; the cap of each case is 2 x its measured count (0 stays 0).  Single-drone cases: none.
MEASURED_ILL = {"m11_g16": 3, "m16_full": 2, "m20_g32": 1, "m2_dyn_euler": 1, "m32_full": 2, "m3_all_aero": 6, "m3_kin20_rpm": 3,
                "m3_multi_hover_obs13": 2, "m4_attitude_kin20": 3, "m4_domain_randomisation_all_aero": 2, "m4_latency_motor_lag_dr": 5,
                "m4_motor_lag_dr_all_aero": 4, "m5_sensors_obs13_dr": 2, "m6_dw_only": 2}      # every other case: 0


def ill_cap(name, w):
    return 2 * MEASURED_ILL.get(name, 0) / w.n_envs + 1e-9


@pytest.mark.parametrize("kernel", ["jit", "generic"])
@pytest.mark.parametrize("name", sorted(CASES))
def test_generic_kernel_parity(name, kernel, monkeypatch):
    """Every case twice: through the run-time instantiation of its feature word (NVRTC), and under MDG_JIT=0 through the
    runtime-flag generic kernel, which is what runs when NVRTC or the sources are not available."""
    w, extra = CASES[name]
    monkeypatch.setenv("MDG_JIT", "1" if kernel == "jit" else "0")
    res = run_parity(w, steps=48, extra=extra, max_ill_frac=ill_cap(name, w))
    print(name, kernel, res)
    assert kernel in res["kernel"], res["kernel"]


@pytest.mark.parametrize("kernel", ["jit", "generic"])
def test_race_airframe_parity(kernel, monkeypatch):
    """Table 2's RACE column (mass 0.25 kg, k_f 1.28e-8): rotor speeds around its own hover RPM (6,920)."""
    monkeypatch.setenv("MDG_JIT", "1" if kernel == "jit" else "0")
    w = wl("race", 1200, 1, W.PHYS_MJC_GND, W.ACT_RPM,
           dict(reset_center=[0, 0, 1], reset_half=[0.1, 0.1, 0.1], reward_mode=W.REW_HOVER, term_mode=W.TERM_HOVER,
                target_mode=W.TGT_FIXED, target_fixed=[0, 0, 1], episode_len_s=10.0, auto_reset=1), ("uniform", 6300.0, 7500.0))
    res = run_parity(w, steps=48, model=W.MODEL_RACE)
    print(res)
    assert kernel in res["kernel"], res["kernel"]


def test_error_paths_and_step_many():
    """Argument errors come back as codes (no abort); a CUDA-graph replay of n steps equals n single steps."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    for bad in [dict(n_envs=0, n_drones=1), dict(n_envs=4, n_drones=33), dict(n_envs=4, n_drones=0)]:
        with pytest.raises(mdg.MdgError):
            mdg.Env(bad["n_envs"], bad["n_drones"], W.PHYS_MJC, W.ACT_RPM)
    with pytest.raises(mdg.MdgError):
        mdg.Env(4, 1, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, sim_freq=250, ctrl_freq=48))   # not a multiple
    w = W.config(5).scaled(3000)
    a, b = (mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **w.params)) for _ in range(2))
    a.reset(w.seed); b.reset(w.seed)
    acts = torch.stack([a.gen_actions(w.seed, t, 1.0, -1.0, 1.0) for t in range(6)])
    with pytest.raises(mdg.MdgError):
        a.step(acts.view(-1)[1:1 + w.n_envs * w.n_drones * 4])                                 # not 16-byte aligned
    for t in range(6):
        a.step(acts[t])
    b.step_many(acts, 6)
    b.step_many(acts, 6)                                                                       # cached graph, replayed
    for t in range(6):
        a.step(acts[t])
    torch.cuda.synchronize()
    sa, sb = a.get_state(), b.get_state()
    assert np.array_equal(sa["state"], sb["state"]) and np.array_equal(sa["ep_step"], sb["ep_step"])
    assert torch.equal(a.obs, b.obs) and torch.equal(a.reward, b.reward) and torch.equal(a.done, b.done)


@pytest.mark.parametrize("kernel", ["jit", "generic"])
@pytest.mark.parametrize("act", [W.ACT_RPM, W.ACT_PID, W.ACT_ATTITUDE])
def test_cf2p_airframe_parity(act, kernel, monkeypatch):
    """The +-configuration mixing: rotor wrench for raw RPMs, the mixer inverse under PID and ATTITUDE."""
    monkeypatch.setenv("MDG_JIT", "1" if kernel == "jit" else "0")
    params = dict(SINGLE)
    actions = HOVER
    if act == W.ACT_PID:
        params.update(reward_mode=W.REW_NEG_SQ_DIST, term_mode=W.TERM_TILT_DIST, term_tilt=0.4, term_dist=3.0,
                      target_mode=W.TGT_BOX, target_lo=[-1, -1, 0.2], target_hi=[1, 1, 2.0])
        actions = ("targets",)
    elif act == W.ACT_ATTITUDE:
        actions = ("uniform", -0.3, 0.3)
    res = run_parity(wl("cf2p", 1100, 1, W.PHYS_MJC_DRAG, act, params, actions), steps=48, model=W.MODEL_CF2P)
    print(res)
    assert kernel in res["kernel"], res["kernel"]


def test_domain_randomisation_factors_match_the_oracle_draws():
    """The factors themselves (Philox streams 4 and 5) after reset and after auto-resets, and mdg_set_dr / mdg_get_dr."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    from oracle import oracle as O
    w = wl("drdraw", 700, 3, W.PHYS_MJC, W.ACT_RPM, dict(GRID, episode_len_s=3 / 48, dr_alpha=DR), HOVER)
    gpu = mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **w.params))
    orc = O.OracleEnv(w.n_envs, w.n_drones, w.physics_mode, w.action_type, O.OracleParams(0, **w.params), n_threads=4)
    gpu.reset(w.seed); orc.reset(w.seed)
    assert np.abs(gpu.get_dr() - orc.dr).max() < 2e-7
    for t in range(7):                                        # truncation every 3 steps -> two redraws
        a = O.gen_actions(w.seed, t, w.n_envs, w.n_drones, W.hover_rpm_f32(), 0.9, 1.1)
        gpu.step(torch.from_numpy(a).cuda()); orc.step(a)
    f = gpu.get_dr()
    assert np.abs(f - orc.dr).max() < 2e-7 and f.std() > 0.01
    f2 = np.ones_like(f); f2[:, 0] = 1.1
    gpu.set_dr(f2)
    assert np.array_equal(gpu.get_dr(), f2)
    plain = mdg.Env(8, 1, W.PHYS_MJC, W.ACT_RPM)
    assert np.all(plain.get_dr() == 1.0)
    with pytest.raises(mdg.MdgError):
        plain.set_dr(np.ones((8, 16), dtype=np.float32))


def test_sensor_noise_residual_and_refresh_after_set_state():
    """Table 4 sensor rows through the C ABI: the noisy handle's state / reward / done are bitwise those of a noise-free handle,
    the residual obs_noisy - obs_clean equals the oracle's residual (same Philox draws), and mdg_set_state recomputes the
    row with the draws of the current step index and episode.  A negative standard deviation is MDG_EINVAL."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    from oracle import oracle as O
    w = wl("sensres", 2000, 2, W.PHYS_MJC_DRAG, W.ACT_RPM, dict(GRID, grid_cols=2, episode_len_s=5 / 48), HOVER)
    noisy_p = dict(w.params, **SENS)
    clean = mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **w.params))
    noisy = mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **noisy_p))
    orc_c = O.OracleEnv(w.n_envs, w.n_drones, w.physics_mode, w.action_type, O.OracleParams(0, **w.params), n_threads=4)
    orc_n = O.OracleEnv(w.n_envs, w.n_drones, w.physics_mode, w.action_type, O.OracleParams(0, **noisy_p), n_threads=4)
    assert "generic" in noisy.kernel_name or "jit" in noisy.kernel_name
    for env in (clean, noisy, orc_c, orc_n):
        env.reset(w.seed)
    for t in range(8):                                                 # truncation after 5 steps: one bias redraw on the way
        if t > 0:
            a = O.gen_actions(w.seed, t, w.n_envs, w.n_drones, W.hover_rpm_f32(), 0.9, 1.1)
            a_dev = torch.from_numpy(a).cuda()
            for env in (clean, noisy):
                env.step(a_dev)
            for env in (orc_c, orc_n):
                env.step(a)
        torch.cuda.synchronize()
        sc, sn = clean.get_state(), noisy.get_state()
        assert np.array_equal(sc["state"], sn["state"]) and np.array_equal(sc["ep_step"], sn["ep_step"])
        assert torch.equal(clean.reward, noisy.reward) and torch.equal(clean.done, noisy.done)
        res32 = (noisy.obs - clean.obs).cpu().numpy().astype(np.float64)
        res64 = orc_n.outputs()[0] - orc_c.outputs()[0]
        assert np.abs(res64).max() > 0.1                               # some 4-sigma draws among 48,000
        assert np.abs(res32 - res64).max() < 2e-6, (t, np.abs(res32 - res64).max())   # fp32 rounding of obs + residual
    # set_state: same state into both sides, other episode counters -> the row uses (gstep, gstep - ep_step)
    st = orc_n.state.astype(np.float32)
    st[:, 0:3] += 0.125
    eps = (np.arange(w.n_envs) % 3).astype(np.uint32)
    orc_n.ep_step = eps
    orc_n.state = st.astype(np.float64)
    noisy.set_state(state=st, ep_step=eps)
    torch.cuda.synchronize()
    assert np.abs(noisy.obs.cpu().numpy() - orc_n.outputs()[0]).max() < 2e-6
    with pytest.raises(mdg.MdgError):
        mdg.Env(4, 1, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, obs_noise=[0.01, -0.05, 0.0, 0.0]))


def test_dryden_altitude_wind_state_matches_the_oracle():
    """The gust state itself under the altitude-dependent length scale: drones parked at hand-picked altitudes (k_wind = 0, hover
    thrust), so alpha(h) is the only thing that shapes the sequence; compared with the oracle's wind after every step."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    from oracle import oracle as O
    N, M = 512, 2
    over = dict(aero_mask=W.AERO_WIND, dryden_airspeed=8.0, k_wind=0.0, wind_sigma=0.7, term_mode=W.TERM_NONE, auto_reset=0, episode_len_s=0.0)
    gpu = mdg.Env(N, M, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, **over))
    orc = O.OracleEnv(N, M, W.PHYS_MJC, W.ACT_RPM, O.OracleParams(0, **over), n_threads=4)
    assert "generic" in gpu.kernel_name or "jit" in gpu.kernel_name
    gpu.reset(9); orc.reset(9)
    st = orc.state.astype(np.float32)
    h = np.linspace(0.01, 3.0, N * M, dtype=np.float32)                # from below the altitude floor to 3 m
    st[:, 0:3] = np.stack([np.arange(N * M) % M * 0.7, np.zeros(N * M), h], axis=1)
    orc.state = st.astype(np.float64)
    gpu.set_state(state=st)
    a = np.full((N * M, 4), W.hover_rpm_f32(), dtype=np.float32)
    a_dev = torch.from_numpy(a).cuda()
    for t in range(24):
        gpu.step(a_dev); orc.step(a)
        w32, w64 = gpu.get_state()["wind"].astype(np.float64), orc.wind
        assert np.abs(w32 - w64).max() < 5e-6, (t, np.abs(w32 - w64).max())
    assert w64.std() > 0.2
    with pytest.raises(mdg.MdgError):
        mdg.Env(4, 1, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, dryden_airspeed=-1.0))


def test_latency_error_paths_and_graph_replay():
    """Latency windows outside what the history planes hold are MDG_EINVAL; a CUDA-graph replay of the latency path equals single steps."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    for over in (dict(act_latency_hi=0.070), dict(obs_latency_hi=0.030), dict(act_latency_lo=0.02, act_latency_hi=0.01), dict(obs_latency_lo=-0.01)):
        with pytest.raises(mdg.MdgError):
            mdg.Env(4, 1, W.PHYS_MJC, W.ACT_RPM, mdg.default_params(0, **over))
    w = wl("latgraph", 3000, 2, W.PHYS_MJC_DRAG, W.ACT_RPM, dict(GRID, grid_cols=2, episode_len_s=0.1, **LAT, **SENS), HOVER)
    a, b = (mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **w.params)) for _ in range(2))
    a.reset(w.seed); b.reset(w.seed)
    acts = torch.stack([a.gen_actions(w.seed, t, W.hover_rpm_f32(), 0.9, 1.1) for t in range(6)])
    for rep in range(2):
        for t in range(6):
            a.step(acts[t])
        b.step_many(acts, 6)
    torch.cuda.synchronize()
    sa, sb = a.get_state(), b.get_state()
    assert np.array_equal(sa["state"], sb["state"]) and np.array_equal(sa["ep_step"], sb["ep_step"])
    assert torch.equal(a.obs, b.obs) and torch.equal(a.reward, b.reward) and torch.equal(a.done, b.done)


def test_async_host_step_on_two_streams_equals_the_synchronous_call():
    """mdg_step_host_async / mdg_wait: two handles double-buffered on two streams produce, bit for bit, what mdg_step_host does."""
    import torch
    import paper_2606_08039_b200 as mdg
    w = W.config(5).scaled(5000)
    mk = lambda base: mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, env_index_base=base)))
    sync = [mk(0), mk(w.n_envs)]
    asy = [mk(0), mk(w.n_envs)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for i in range(2):
        asy[i].set_stream(streams[i])
        sync[i].reset(w.seed); asy[i].reset(w.seed)
    torch.cuda.synchronize()
    acts = [[sync[i].gen_actions(w.seed, t, 1.0, -1.0, 1.0).cpu().pin_memory() for t in range(5)] for i in range(2)]
    def bufs():
        return (torch.empty((w.n_envs, sync[0].obs_dim)).pin_memory(), torch.empty(w.n_envs).pin_memory(), torch.empty(w.n_envs, dtype=torch.uint8).pin_memory())
    bs, ba = [bufs(), bufs()], [bufs(), bufs()]
    for t in range(5):
        for i in range(2):
            sync[i].step_host(acts[i][t], *bs[i])
        asy[0].step_host(acts[0][t], *ba[0], asynchronous=True)
        asy[1].step_host(acts[1][t], *ba[1], asynchronous=True)
        asy[0].wait(); asy[1].wait()
        for i in range(2):
            for x, y in zip(bs[i], ba[i]):
                assert torch.equal(x, y), (t, i)
    assert bs[0][0].abs().max() > 0.1 and not torch.equal(bs[0][0], bs[1][0])


def test_formation_path_targets_follow_the_oracle_and_bad_paths_are_rejected():
    """mdg_targets under the moving formation centre: the slots of the moment, step by step, across a lap and an auto-reset."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    from oracle import oracle as O
    w = wl("pathtg", 64, 3, W.PHYS_MJC, W.ACT_VEL,
           dict(CIRCLE, target_mode=W.TGT_CIRCLE, episode_len_s=1.0, form_path_n=3, form_speed=4.0, form_path=[0, 0, 1, 0.5, 0.1, 1.2, 0.2, 0.6, 0.9] + [0.0] * 15),
           ("uniform", -0.2, 0.2))
    gpu = mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **w.params))
    orc = O.OracleEnv(w.n_envs, w.n_drones, w.physics_mode, w.action_type, O.OracleParams(0, **w.params))
    assert "generic" in gpu.kernel_name or "jit" in gpu.kernel_name
    gpu.reset(w.seed); orc.reset(w.seed)
    seen = []
    for t in range(60):                                                # perimeter 1.74 m at 4 m/s: two laps; truncation after 48 steps
        a = O.gen_actions(w.seed, t, w.n_envs, w.n_drones, 1.0, -0.2, 0.2)
        gpu.step(torch.from_numpy(a).cuda()); orc.step(a)
        tg = gpu.get_state()["targets"].astype(np.float64)
        assert np.abs(tg[:, :3] - orc.targets[:, :3]).max() < 2e-6, t
        seen.append(tg[0, :3].copy())
    assert np.ptp(np.array(seen), axis=0).min() > 0.25                 # the slot really travelled
    for over in (dict(form_path_n=9), dict(form_path_n=-1), dict(form_speed=-1.0)):
        with pytest.raises(mdg.MdgError):
            mdg.Env(4, 2, W.PHYS_MJC, W.ACT_VEL, mdg.default_params(0, **dict(w.params, **over)))


def test_checkpoint_resume_is_bitwise_with_every_stateful_feature_on():
    """mdg_save / mdg_load: DR factors, rotor speeds, gust impulses, action history, counters, seed and outputs travel in the blob;
    a second handle that loads it continues exactly like the first (chained steps and a graph replay included)."""
    import numpy as np
    import torch
    import paper_2606_08039_b200 as mdg
    w = wl("ckpt", 3000, 4, W.PHYS_MJC_GND_DRAG_DW, W.ACT_RPM,
           dict(GRID, grid_cols=2, episode_len_s=0.3, aero_mask=15, wind_mask=15, wind_const=[0.0, 0.9, 0.0], wind_sine_amp=0.01, wind_sine_omega=3.0,
                gust_prob=0.2, gust_max=1.5, gust_duration=0.3, dryden_airspeed=6.0, dr_alpha=DR, motor_lag_lo=0.005, motor_lag_hi=0.05, **INIT, **LAT, **SENS), HOVER)
    mk = lambda: mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type, mdg.default_params(0, **w.params))
    a, b = mk(), mk()
    a.reset(w.seed); b.reset(12345)
    acts = [a.gen_actions(w.seed, t, W.hover_rpm_f32(), 0.9, 1.1) for t in range(30)]
    for t in range(14):
        a.step(acts[t])
    blob = a.save()
    for t in range(14):
        b.step(acts[t])                                                # b is somewhere else entirely when the blob arrives
    b.load(blob)
    assert torch.equal(a.obs, b.obs) and torch.equal(a.reward, b.reward) and torch.equal(a.done, b.done)
    for t in range(14, 24):
        a.step(acts[t]); b.step(acts[t])
    stack = torch.stack(acts[24:30])
    a.step_many(stack, 6); b.step_many(stack, 6)
    torch.cuda.synchronize()
    sa, sb = a.get_state(), b.get_state()
    for k in sa:
        assert np.array_equal(sa[k], sb[k]), k
    assert np.array_equal(a.get_dr(), b.get_dr())
    assert torch.equal(a.obs, b.obs) and torch.equal(a.reward, b.reward) and torch.equal(a.done, b.done)
    assert torch.equal(a.reward_per_drone, b.reward_per_drone)
    assert np.array_equal(a.save(), b.save())
    # error paths: another shape, another feature set, a truncated or foreign blob
    other = mdg.Env(w.n_envs, 2, w.physics_mode, w.action_type, mdg.default_params(0, **dict(w.params, grid_cols=2)))
    plain = mdg.Env(w.n_envs, w.n_drones, w.physics_mode, w.action_type)
    for env, data in ((other, blob), (plain, blob), (b, blob[:1000]), (b, blob[: blob.size - 8]), (b, np.zeros(blob.size, dtype=np.uint8))):
        with pytest.raises(mdg.MdgError):
            env.load(data)


@pytest.mark.parametrize("variant,tag", [("dyn", ",dyn>"), ("table4", ",table4>")])
def test_config5_variant_specialisations_parity(variant, tag):
    """The two extra compile-time specialisations on the metric's config (bench.py --variant): Table 1's DYN integrator, and every
    row of Table 4 on (DR factors, motor lag, action / sensor latency, sensor noise) - same parity bar as config 5 itself."""
    # exactly the overrides bench.py --variant times (workloads.VARIANTS), plus short episodes so that the per-episode draws recur
    over = dict(W.VARIANTS[variant], **({"episode_len_s": 0.4} if variant == "table4" else {}))
    w = W.config(5).scaled(4099)
    res = run_parity(w, steps=48, extra=over, max_ill_frac=0.0)
    print(variant, res)
    assert tag[:-1] in res["kernel"], res["kernel"]


def test_paper_mjx_workload_specialisation_parity():
    """HoverAviary as the paper's MJX back end runs it (rigid body only, normalised rotor commands PAPER.md:300):
    its own compile-time specialisation (bench.py --variant paper_mjx)."""
    res = run_parity(wl("mjx", 4099, 1, W.PHYS_MJC, W.ACT_RPM_NORM, dict(SINGLE), ("uniform", -0.05, 0.06)), steps=48)
    print(res)
    assert res["kernel"].startswith("step_kernel<G=1,rigid,rpm_norm,hover")


def test_run_time_specialisation_and_generic_fallback_agree_with_the_oracle(monkeypatch):
    """A feature word without a precompiled specialisation is instantiated at mdg_create (NVRTC over the same source); MDG_JIT=0
    keeps the runtime-flag generic kernel.  Both must meet the parity bar on the same workload."""
    w, extra = CASES["m4_wind_combined_c5_like"]
    res = run_parity(w, steps=24, extra=extra, max_ill_frac=0.0)
    assert "jit" in res["kernel"], res["kernel"]
    monkeypatch.setenv("MDG_JIT", "0")
    res0 = run_parity(w, steps=24, extra=extra, max_ill_frac=0.0)
    assert "generic" in res0["kernel"], res0["kernel"]

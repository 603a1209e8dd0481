"""ctypes front end of the float64 CPU oracle (TEST INFRASTRUCTURE, see drone_oracle.hpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this.  It never imports the product package and the product never imports it.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        L.orc_params_new.restype = C.c_void_p
        L.orc_params_new.argtypes = [C.c_int]
        L.orc_params_free.argtypes = [C.c_void_p]
        L.orc_params_set.argtypes = [C.c_void_p, C.c_char_p, C.c_int, C.c_double]
        L.orc_params_get.argtypes = [C.c_void_p, C.c_char_p, C.c_int, C.POINTER(C.c_double)]
        L.orc_derived.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_obs_dim.argtypes = [C.c_void_p]
        L.orc_reset.argtypes = [C.c_void_p, C.c_uint64]
        L.orc_step.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.orc_flop_tally.restype = C.c_uint64
        L.orc_flop_tally.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_flop_parts.argtypes = [C.c_void_p]
        L.orc_count_flops.restype = C.c_uint64
        L.orc_count_flops.argtypes = [C.c_char_p]
        for n in ("state", "pid", "targets", "wind", "ep_step", "dr", "gust", "rotor"):
            getattr(L, "orc_get_" + n).argtypes = [C.c_void_p, C.c_void_p]
            getattr(L, "orc_set_" + n).argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_gstep.restype = C.c_uint32
        L.orc_get_gstep.argtypes = [C.c_void_p]
        L.orc_get_outputs.argtypes = [C.c_void_p] * 5
        L.orc_get_reward_d.argtypes = [C.c_void_p] * 2
        L.orc_refresh_obs.argtypes = [C.c_void_p]
        L.orc_probe_wrench.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_probe_decode.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_motor_wrench.argtypes = [C.c_void_p] * 3
        L.orc_alloc_inverse.argtypes = [C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_euler_zyx.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_quat_exp_step.argtypes = [C.c_void_p] * 3
        L.orc_philox.argtypes = [C.c_uint32] * 6 + [C.c_void_p]
        L.orc_wind_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_gen_actions.argtypes = [C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, C.c_void_p, C.c_uint32]
        L.orc_render_depth.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_render_rgba.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.c_void_p] * 6 + [C.c_int]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class OracleParams:
    """Name-keyed parameter block (defaults: Table 2 / Table 6 + the readings of DESIGN.md §3)."""

    def __init__(self, model=0, **overrides):
        self._h = lib().orc_params_new(model)
        self.update(overrides)

    def update(self, d):
        for k, v in d.items():
            self[k] = v
        return self

    def __setitem__(self, name, value):
        vals = np.atleast_1d(np.asarray(value, dtype=np.float64))
        for i, v in enumerate(vals):
            if lib().orc_params_set(self._h, name.encode(), i, float(v)) != 0:
                raise KeyError(f"oracle params: no field {name}[{i}]")

    def get(self, name, idx=0):
        out = C.c_double()
        if lib().orc_params_get(self._h, name.encode(), idx, C.byref(out)) != 0:
            raise KeyError(name)
        return out.value

    def derived(self, physics_mode=0):
        out = np.zeros(12)
        lib().orc_derived(self._h, physics_mode, _p(out))
        keys = ["W", "hover_rpm", "max_rpm", "l", "kappa", "s_max", "h", "dt_c", "K", "ep_steps", "aero", "integ"]
        return dict(zip(keys, out.tolist()))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_params_free(self._h)
            self._h = None


FLOP_PHASES = ("wind", "decode", "motor", "wrench", "integrate", "obs", "reward")


def count_flops(name):
    """Flops of one call of a building block of the oracle on its counting scalar (oracle_capi.cpp: orc_count_flops)."""
    n = int(lib().orc_count_flops(name.encode()))
    if n == 2 ** 64 - 1:
        raise KeyError(name)
    return n


class OracleEnv:
    """The batched env of SURVEY.md §8(b) computed by the float64 oracle."""

    def __init__(self, n_envs, n_drones, physics_mode, action_type, params: OracleParams, n_threads=1):
        self.N, self.M = n_envs, n_drones
        self.params = params
        self.n_threads = n_threads
        self._h = lib().orc_create(n_envs, n_drones, physics_mode, action_type, params._h)
        if not self._h:
            raise ValueError("oracle: invalid arguments")
        self.obs_dim = lib().orc_obs_dim(self._h)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def reset(self, seed):
        lib().orc_reset(self._h, int(seed))

    def step(self, actions):
        a = np.ascontiguousarray(actions, dtype=np.float32).reshape(-1)
        assert a.size == self.N * self.M * 4
        lib().orc_step(self._h, _p(a), self.n_threads)

    def flop_tally(self, actions):
        a = np.ascontiguousarray(actions, dtype=np.float32).reshape(-1)
        assert a.size == self.N * self.M * 4
        return int(lib().orc_flop_tally(self._h, _p(a)))

    def flop_parts(self, actions):
        """The tally of flop_tally(actions) by phase of the control step (drone_oracle.hpp: PH_*)."""
        total = self.flop_tally(actions)
        out = np.zeros(len(FLOP_PHASES), dtype=np.uint64)
        lib().orc_flop_parts(_p(out))
        assert int(out.sum()) == total
        return dict(zip(FLOP_PHASES, (int(x) for x in out)))

    def _get(self, name, shape, dtype=np.float64):
        out = np.zeros(shape, dtype=dtype)
        getattr(lib(), "orc_get_" + name)(self._h, _p(out))
        return out

    def _set(self, name, arr, shape, dtype=np.float64):
        a = np.ascontiguousarray(arr, dtype=dtype).reshape(shape)
        getattr(lib(), "orc_set_" + name)(self._h, _p(a))

    @property
    def state(self):            # [N*M, 13] = p(3) q(4, wxyz) v(3) w_body(3)
        return self._get("state", (self.N * self.M, 13))

    @state.setter
    def state(self, v):
        self._set("state", v, (self.N * self.M, 13))
        lib().orc_refresh_obs(self._h)

    @property
    def pid(self):              # [N*M, 10] = I_p(3) I_eta(3) held setpoint(4)
        return self._get("pid", (self.N * self.M, 10))

    @pid.setter
    def pid(self, v):
        self._set("pid", v, (self.N * self.M, 10))

    @property
    def targets(self):          # [N*M, 4]
        return self._get("targets", (self.N * self.M, 4))

    @targets.setter
    def targets(self, v):
        self._set("targets", v, (self.N * self.M, 4))

    @property
    def wind(self):             # [N, 3]
        return self._get("wind", (self.N, 3))

    @wind.setter
    def wind(self, v):
        self._set("wind", v, (self.N, 3))

    @property
    def dr(self):               # [N*M, 16] DR factors [m, J, k_f, k_m, drag, C_gnd, C_1, g, motor bias x4, arm, MAX_RPM, 1, 1]
        return self._get("dr", (self.N * self.M, 16))

    @dr.setter
    def dr(self, v):
        self._set("dr", v, (self.N * self.M, 16))

    @property
    def ep_step(self):
        return self._get("ep_step", (self.N,), np.uint32)

    @ep_step.setter
    def ep_step(self, v):
        self._set("ep_step", v, (self.N,), np.uint32)

    @property
    def gstep(self):
        return int(lib().orc_get_gstep(self._h))

    def outputs(self):
        obs = np.zeros((self.N, self.obs_dim))
        rew = np.zeros(self.N)
        done = np.zeros(self.N, dtype=np.uint8)
        margin = np.zeros((self.N, 3))
        lib().orc_get_outputs(self._h, _p(obs), _p(rew), _p(done), _p(margin))
        return obs, rew, done, margin

    @property
    def rotor(self):            # [N*M, 4] rotor speeds actually turning (RPM): the state of the motor lag
        return self._get("rotor", (self.N * self.M, 4))

    @rotor.setter
    def rotor(self, v):
        self._set("rotor", v, (self.N * self.M, 4))

    @property
    def gust(self):             # [N, 4] running gust impulse: velocity vector and progress s (>= 1: none)
        return self._get("gust", (self.N, 4))

    @gust.setter
    def gust(self, v):
        self._set("gust", v, (self.N, 4))

    @property
    def reward_per_drone(self):   # [N*M] per-drone share of the last step's reward (sums to the env reward)
        return self._get("reward_d", (self.N * self.M,))

    def probe_wrench(self, env, rpm):
        rpm = _f64(rpm).reshape(self.M, 4)
        F = np.zeros((self.M, 3))
        tau = np.zeros((self.M, 3))
        lib().orc_probe_wrench(self._h, env, _p(rpm), _p(F), _p(tau))
        return F, tau

    def probe_decode(self, actions, commit=False):
        a = np.ascontiguousarray(actions, dtype=np.float32).reshape(-1)
        assert a.size == self.N * self.M * 4
        rpm = np.zeros((self.N * self.M, 4))
        lib().orc_probe_decode(self._h, _p(a), _p(rpm), int(commit))
        return rpm


def motor_wrench(params, rpm):
    rpm = _f64(rpm).reshape(4)
    out = np.zeros(5)
    lib().orc_motor_wrench(params._h, _p(rpm), _p(out))
    return out[0], out[1:4].copy(), out[4]


def alloc_inverse(params, T, tau):
    tau = _f64(tau).reshape(3)
    s = np.zeros(4)
    lib().orc_alloc_inverse(params._h, float(T), _p(tau), _p(s))
    return s


def euler_zyx(q):
    q = _f64(q).reshape(4)
    eta = np.zeros(3)
    lib().orc_euler_zyx(_p(q), _p(eta))
    return eta


def quat_exp_step(q, phi):
    q = _f64(q).reshape(4)
    phi = _f64(phi).reshape(3)
    out = np.zeros(4)
    lib().orc_quat_exp_step(_p(q), _p(phi), _p(out))
    return out


def philox(counter, key):
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(*[int(c) for c in counter], int(key[0]), int(key[1]), _p(out))
    return out


def wind_normals(seed, env, t):
    xi = np.zeros(3)
    lib().orc_wind_normals(int(seed), int(env), int(t), _p(xi))
    return xi


def gen_actions(seed, t, n_envs, n_drones, base, lo, hi, env_base=0):
    """Harness actions for control step t (Philox stream 3): base * (lo + (hi-lo) u), fp32 [N*M, 4]."""
    out = np.zeros((n_envs * n_drones, 4), dtype=np.float32)
    lib().orc_gen_actions(int(seed), int(t), n_envs, n_drones, float(base), float(lo), float(hi), _p(out), int(env_base))
    return out


# NEXT-4 camera (camera_oracle.hpp; readings Q45-Q48).  body_a = arm + propeller radius of CF2X (Table 2), body_c = reading Q46.
CAM_DEFAULTS = dict(H=48, W=64, fovy_deg=60.0, offset=(0.02, 0.0, 0.0), znear=0.01, zfar=50.0, body_a=0.0397 + 0.02325, body_c=0.0125)


def render_depth(state, n_envs, n_drones, n_threads=1, with_margin=False, **cam):
    """Depth [D, H, W] float64 and segmentation [D, H, W] u8 of every drone's camera from state [D, 13] (float64)."""
    c = dict(CAM_DEFAULTS)
    for k in cam:
        if k not in c:
            raise KeyError(k)
    c.update(cam)
    st = _f64(state).reshape(n_envs * n_drones, 13)
    H, W = int(c["H"]), int(c["W"])
    vec = np.array([H, W, c["fovy_deg"], *c["offset"], c["znear"], c["zfar"], c["body_a"], c["body_c"]], dtype=np.float64)
    D = n_envs * n_drones
    depth = np.empty((D, H, W), np.float64)
    seg = np.empty((D, H, W), np.uint8)
    margin = np.empty((D, H, W), np.float64) if with_margin else None
    lib().orc_render_depth(_p(st), n_envs, n_drones, _p(vec), _p(depth), _p(seg), _p(margin) if with_margin else None, int(n_threads))
    return (depth, seg, margin) if with_margin else (depth, seg)


def render_rgba(state, n_envs, n_drones, n_threads=1, **cam):
    """The colour frame of reading Q53 (camera_oracle.hpp): rgba [D, H, W, 4] u8, with depth, segmentation, the tie margin of
    the hit decisions and the shade before quantisation (1 for the background), all [D, H, W]."""
    c = dict(CAM_DEFAULTS)
    for k in cam:
        if k not in c:
            raise KeyError(k)
    c.update(cam)
    st = _f64(state).reshape(n_envs * n_drones, 13)
    H, W = int(c["H"]), int(c["W"])
    vec = np.array([H, W, c["fovy_deg"], *c["offset"], c["znear"], c["zfar"], c["body_a"], c["body_c"]], dtype=np.float64)
    D = n_envs * n_drones
    depth, seg, margin = np.empty((D, H, W), np.float64), np.empty((D, H, W), np.uint8), np.empty((D, H, W), np.float64)
    rgba, sm = np.empty((D, H, W, 4), np.uint8), np.empty((D, H, W), np.float64)
    lib().orc_render_rgba(_p(st), n_envs, n_drones, _p(vec), _p(depth), _p(seg), _p(margin), _p(rgba), _p(sm), int(n_threads))
    return rgba, depth, seg, margin, sm

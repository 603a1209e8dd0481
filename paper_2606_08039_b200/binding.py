"""Thin ctypes binding of libmdg.so — argument marshalling only; every step of the path runs in the
CUDA kernels behind the C ABI of include/mdg.h.  Function names mirror the C names (mdg_step -> step).
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmdg.so")
STATIC_STAGE_MAX_DRONES = 262144     # include/mdg.h: MDG_STATIC_STAGE_MAX_DRONES

MDG_OK, MDG_EINVAL, MDG_ECUDA, MDG_ENOMEM = 0, -1, -2, -3


class mdg_params(C.Structure):
    """Mirror of `struct mdg_params` (include/mdg.h)."""
    _F3 = C.c_float * 3
    _fields_ = [
        ("struct_size", C.c_uint32), ("drone_model", C.c_int32),
        ("m", C.c_float), ("g", C.c_float), ("L", C.c_float), ("k_f", C.c_float), ("k_m", C.c_float),
        ("J", _F3), ("r_p", C.c_float), ("tw_ratio", C.c_float),
        ("C_gnd", C.c_float), ("h_clip", C.c_float), ("c_xy", C.c_float), ("c_z", C.c_float),
        ("dw_C1", C.c_float), ("dw_C2", C.c_float), ("dw_C3", C.c_float), ("dw_dz_clip", C.c_float),
        ("k_wind", C.c_float), ("wind_sigma", C.c_float), ("wind_tau", C.c_float),
        ("sim_freq", C.c_int32), ("ctrl_freq", C.c_int32), ("aero_mask", C.c_int32), ("integrator", C.c_int32),
        ("Kp_pos", _F3), ("Ki_pos", _F3), ("Kd_pos", _F3), ("Kp_att", _F3), ("Ki_att", _F3), ("Kd_att", _F3),
        ("int_clamp_pos", C.c_float), ("int_clamp_att", C.c_float), ("dsl", C.c_int32),
        ("pos_rate_limit", C.c_float), ("yaw_rate_limit", C.c_float), ("a_ff", _F3),
        ("tilt_max", C.c_float), ("tau_xy_max", C.c_float), ("tau_z_max", C.c_float),
        ("obs_mode", C.c_int32), ("adj_radius", C.c_float), ("reward_mode", C.c_int32), ("at_target_radius", C.c_float),
        ("term_mode", C.c_int32), ("term_tilt", C.c_float), ("term_dist", C.c_float), ("term_center", _F3), ("z_max", C.c_float),
        ("episode_len_s", C.c_float), ("auto_reset", C.c_int32),
        ("reset_layout", C.c_int32), ("reset_center", _F3), ("reset_half", _F3), ("reset_z_lo", C.c_float), ("reset_z_hi", C.c_float),
        ("grid_cols", C.c_int32), ("grid_spacing", C.c_float), ("circle_radius", C.c_float),
        ("target_mode", C.c_int32), ("target_fixed", _F3), ("target_lo", _F3), ("target_hi", _F3),
        ("mh_z_lo", C.c_float), ("mh_z_hi", C.c_float), ("form_center", _F3), ("form_radius", C.c_float),
        ("env_index_base", C.c_uint32), ("target_w_lo", C.c_float), ("target_w_hi", C.c_float), ("dr_alpha", C.c_float * 12), ("reset_rpy_half", _F3), ("reset_vel_half", _F3), ("motor_lag_lo", C.c_float), ("motor_lag_hi", C.c_float),
        ("wind_mask", C.c_int32), ("wind_const", _F3), ("wind_sine_amp", C.c_float), ("wind_sine_omega", C.c_float),
        ("gust_prob", C.c_float), ("gust_max", C.c_float), ("gust_duration", C.c_float),
        ("n_waypoints", C.c_int32), ("waypoints", C.c_float * 24), ("wp_radius", C.c_float),
        ("wp_bonus", C.c_float), ("wp_shaping", C.c_float), ("wp_speed", C.c_float), ("wp_omega", C.c_float), ("wp_laps", C.c_int32),
        ("obs_noise", C.c_float * 4), ("obs_bias", C.c_float * 4),
        ("dryden_airspeed", C.c_float), ("dryden_h_min", C.c_float),
        ("act_latency_lo", C.c_float), ("act_latency_hi", C.c_float), ("obs_latency_lo", C.c_float), ("obs_latency_hi", C.c_float),
        ("form_path_n", C.c_int32), ("form_path", C.c_float * 24), ("form_speed", C.c_float),
    ]

    def update(self, d):
        for k, v in d.items():
            cur = getattr(self, k)          # raises AttributeError on an unknown field
            if isinstance(cur, C.Array):
                for i, x in enumerate(v):
                    cur[i] = x
            else:
                setattr(self, k, v)
        return self


class mdg_cam_params(C.Structure):
    """Mirror of `struct mdg_cam_params` (include/mdg.h)."""
    _fields_ = [("struct_size", C.c_uint32), ("height", C.c_int32), ("width", C.c_int32), ("fovy_deg", C.c_float),
                ("offset", C.c_float * 3), ("znear", C.c_float), ("zfar", C.c_float),
                ("body_radius", C.c_float), ("body_half_height", C.c_float)]
    update = mdg_params.update


EXPORTS = ["mdg_default_params", "mdg_create", "mdg_destroy", "mdg_reset", "mdg_step", "mdg_step_chained", "mdg_step_many", "mdg_step_host", "mdg_step_host_async", "mdg_step_host_static", "mdg_wait", "mdg_checkpoint_size", "mdg_save", "mdg_load", "mdg_outputs",
           "mdg_obs_dim", "mdg_targets", "mdg_gen_actions", "mdg_get_state", "mdg_set_state", "mdg_set_stream",
           "mdg_launch_count", "mdg_kernel_name", "mdg_set_launch", "mdg_measure_fp32_peak", "mdg_get_dr", "mdg_set_dr", "mdg_reward_per_drone", "mdg_default_cam_params", "mdg_render_depth", "mdg_render_rgba", "mdg_last_error", "mdg_version"]

_lib = None


def lib():
    """Load libmdg.so; fails loudly when the CUDA extension has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_08039_b200.build` "
                               "(nvcc, sm_100a). There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        vp, PP = C.c_void_p, C.POINTER(mdg_params)
        L.mdg_default_params.argtypes = [C.c_int, PP]
        L.mdg_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, PP, C.POINTER(vp)]
        L.mdg_destroy.argtypes = [vp]
        L.mdg_destroy.restype = None
        L.mdg_reset.argtypes = [vp, C.c_uint64]
        L.mdg_step.argtypes = [vp, vp]
        L.mdg_step_chained.argtypes = [vp, vp]
        L.mdg_step_many.argtypes = [vp, vp, C.c_int, C.c_int64]
        L.mdg_step_host.argtypes = [vp] * 5
        L.mdg_step_host_async.argtypes = [vp] * 5
        L.mdg_step_host_static.argtypes = [vp] * 5
        L.mdg_wait.argtypes = [vp]
        L.mdg_checkpoint_size.argtypes = [vp]
        L.mdg_checkpoint_size.restype = C.c_int64
        L.mdg_save.argtypes = [vp, vp, C.c_int64]
        L.mdg_load.argtypes = [vp, vp, C.c_int64]
        L.mdg_outputs.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.mdg_obs_dim.argtypes = [vp]
        L.mdg_targets.argtypes = [vp, C.POINTER(vp)]
        L.mdg_gen_actions.argtypes = [vp, C.c_uint64, C.c_uint32, C.c_float, C.c_float, C.c_float, vp]
        L.mdg_get_state.argtypes = [vp] * 6
        L.mdg_set_state.argtypes = [vp] * 6
        L.mdg_set_stream.argtypes = [vp, vp]
        L.mdg_reward_per_drone.argtypes = [vp, C.POINTER(vp)]
        L.mdg_get_dr.argtypes = [vp, vp]
        L.mdg_set_dr.argtypes = [vp, vp]
        L.mdg_launch_count.argtypes = [vp]
        L.mdg_launch_count.restype = C.c_int64
        L.mdg_kernel_name.argtypes = [vp]
        L.mdg_kernel_name.restype = C.c_char_p
        L.mdg_set_launch.argtypes = [vp, C.c_int, C.c_int]
        L.mdg_last_error.restype = C.c_char_p
        L.mdg_measure_fp32_peak.argtypes = [vp, C.POINTER(C.c_double)]
        L.mdg_default_cam_params.argtypes = [PP, C.POINTER(mdg_cam_params)]
        L.mdg_render_depth.argtypes = [vp, C.POINTER(mdg_cam_params), vp, vp]
        L.mdg_render_rgba.argtypes = [vp, C.POINTER(mdg_cam_params), vp]
        _lib = L
    return _lib


def measure_fp32_peak(stream=None) -> float:
    """Achieved FP32 FFMA rate of the current device in TFLOP/s (include/mdg.h: mdg_measure_fp32_peak)."""
    import torch
    out = C.c_double(0.0)
    s = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().mdg_measure_fp32_peak(C.c_void_p(s.cuda_stream), C.byref(out)))
    return out.value


class MdgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mdg error {code}: {msg}")
        self.code = code


def _check(rc):
    if rc != MDG_OK:
        raise MdgError(rc, lib().mdg_last_error().decode())


def default_params(drone_model=0, **overrides) -> mdg_params:
    p = mdg_params()
    _check(lib().mdg_default_params(drone_model, C.byref(p)))
    return p.update(overrides)


def default_cam_params(params: mdg_params = None, **overrides) -> mdg_cam_params:
    c = mdg_cam_params()
    _check(lib().mdg_default_cam_params(C.byref(params) if params is not None else None, C.byref(c)))
    return c.update(overrides)


class _DevArray:
    """Zero-copy view of library-owned device memory for torch.as_tensor (CUDA array interface v3)."""

    def __init__(self, ptr, shape, typestr, owner):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 3, "strides": None}
        self._owner = owner


class Env:
    """create / reset / step of the batched drone env on the current CUDA device.

    PyTorch supplies device memory and streams only: `step(actions)` takes a CUDA float32 tensor of
    shape [n_envs*n_drones, 4] (or anything reshapeable to it) and `obs`, `reward`, `done` are zero-copy
    tensor views of the library's output buffers.
    """

    def __init__(self, n_envs, n_drones, physics_mode, action_type, params: mdg_params = None, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_08039_b200 needs a CUDA device: there is no CPU fallback")
        self._torch = torch
        self.n_envs, self.n_drones = n_envs, n_drones
        self.params = params if params is not None else default_params()
        h = C.c_void_p()
        _check(lib().mdg_create(n_envs, n_drones, physics_mode, action_type, C.byref(self.params), C.byref(h)))
        self._h = h
        self.obs_dim = lib().mdg_obs_dim(h)
        o, r, d, t = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(lib().mdg_outputs(h, C.byref(o), C.byref(r), C.byref(d)))
        _check(lib().mdg_targets(h, C.byref(t)))
        dev = torch.device("cuda", torch.cuda.current_device())
        self.obs = torch.as_tensor(_DevArray(o.value, (n_envs, self.obs_dim), "<f4", self), device=dev)
        self.reward = torch.as_tensor(_DevArray(r.value, (n_envs,), "<f4", self), device=dev)
        self.done = torch.as_tensor(_DevArray(d.value, (n_envs,), "|u1", self), device=dev)
        self.targets = torch.as_tensor(_DevArray(t.value, (n_envs * n_drones, 4), "<f4", self), device=dev)
        rd = C.c_void_p()
        _check(lib().mdg_reward_per_drone(self._h, C.byref(rd)))
        self.reward_per_drone = torch.as_tensor(_DevArray(rd.value, (n_envs * n_drones,), "<f4", self), device=dev)
        self.set_stream(stream if stream is not None else torch.cuda.current_stream())

    def close(self):
        if getattr(self, "_h", None):
            lib().mdg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        _check(lib().mdg_set_stream(self._h, C.c_void_p(stream.cuda_stream)))

    def set_launch(self, block_threads=0, max_blocks_per_sm=0):
        _check(lib().mdg_set_launch(self._h, block_threads, max_blocks_per_sm))

    def reset(self, seed):
        _check(lib().mdg_reset(self._h, int(seed)))
        return self.obs

    def _act_ptr(self, actions, steps=1):
        t = self._torch
        if not (isinstance(actions, t.Tensor) and actions.is_cuda and actions.dtype == t.float32 and actions.is_contiguous()):
            raise TypeError("actions must be a contiguous CUDA float32 tensor")
        if actions.numel() != steps * self.n_envs * self.n_drones * 4:
            raise ValueError("actions must hold n_envs*n_drones*4 floats per step")
        return C.c_void_p(actions.data_ptr())

    def step(self, actions):
        _check(lib().mdg_step(self._h, self._act_ptr(actions)))
        return self.obs, self.reward, self.done

    def step_chained(self, actions):
        """mdg_step_chained: `actions` must have been complete before the previous step of this env was enqueued (include/mdg.h)."""
        _check(lib().mdg_step_chained(self._h, self._act_ptr(actions)))
        return self.obs, self.reward, self.done

    def step_many(self, actions, n_steps):
        """n_steps control steps replayed as one CUDA graph; actions: [n_steps, n_envs*n_drones, 4]."""
        _check(lib().mdg_step_many(self._h, self._act_ptr(actions, n_steps), n_steps, self.n_envs * self.n_drones * 4))
        return self.obs, self.reward, self.done

    def step_host(self, actions_host, obs_host=None, reward_host=None, done_host=None, asynchronous=False):
        """End-to-end step on HOST tensors (ideally pinned): H2D actions, step, D2H outputs, synchronise.
        asynchronous=True only enqueues (mdg_step_host_async); call wait() before reading the host tensors."""
        def ptr(x):
            return C.c_void_p(None) if x is None else C.c_void_p(x.data_ptr())
        if actions_host.is_cuda or actions_host.numel() != self.n_envs * self.n_drones * 4:
            raise ValueError("actions_host must be a host float32 tensor of n_envs*n_drones*4 elements")
        fn = lib().mdg_step_host_async if asynchronous else lib().mdg_step_host
        _check(fn(self._h, ptr(actions_host), ptr(obs_host), ptr(reward_host), ptr(done_host)))

    def step_host_static(self, actions_host, obs_host=None, reward_host=None, done_host=None):
        """step_host without any allocation: the actions are staged in the library's static device array (mdg_step_host_static;
        at most STATIC_STAGE_MAX_DRONES drones per handle, one array per GPU shared by all handles)."""
        def ptr(x):
            return C.c_void_p(None) if x is None else C.c_void_p(x.data_ptr())
        if actions_host.is_cuda or actions_host.numel() != self.n_envs * self.n_drones * 4:
            raise ValueError("actions_host must be a host float32 tensor of n_envs*n_drones*4 elements")
        _check(lib().mdg_step_host_static(self._h, ptr(actions_host), ptr(obs_host), ptr(reward_host), ptr(done_host)))

    def save(self):
        """Full checkpoint as a numpy uint8 array (include/mdg.h: mdg_save)."""
        import numpy as np
        n = lib().mdg_checkpoint_size(self._h)
        if n < 0:
            _check(int(n))
        buf = np.empty(int(n), dtype=np.uint8)
        _check(lib().mdg_save(self._h, C.c_void_p(buf.ctypes.data), int(n)))
        return buf

    def load(self, blob):
        """Restore a checkpoint written by save() on a handle of the same shape and parameters (mdg_load)."""
        import numpy as np
        b = np.ascontiguousarray(blob, dtype=np.uint8)
        _check(lib().mdg_load(self._h, C.c_void_p(b.ctypes.data), int(b.size)))

    def wait(self):
        """Block until everything enqueued on this handle's stream has finished (include/mdg.h: mdg_wait)."""
        _check(lib().mdg_wait(self._h))

    def gen_actions(self, seed, t, base, lo, hi, out=None):
        if out is None:
            out = self._torch.empty((self.n_envs * self.n_drones, 4), dtype=self._torch.float32, device=self.obs.device)
        _check(lib().mdg_gen_actions(self._h, int(seed), int(t), float(base), float(lo), float(hi), C.c_void_p(out.data_ptr())))
        return out

    def render_depth(self, cam: mdg_cam_params = None, depth=None, seg=None, want_depth=True, want_seg=True):
        """Every drone's onboard camera from the current state (include/mdg.h: mdg_render_depth): depth [D, H, W] float32 and
        segmentation [D, H, W] uint8 CUDA tensors (allocated here unless passed in)."""
        t = self._torch
        c = cam if cam is not None else default_cam_params(self.params)
        shape = (self.n_envs * self.n_drones, c.height, c.width)
        if depth is None and want_depth:
            depth = t.empty(shape, dtype=t.float32, device=self.obs.device)
        if seg is None and want_seg:
            seg = t.empty(shape, dtype=t.uint8, device=self.obs.device)
        for x, dt in ((depth, t.float32), (seg, t.uint8)):
            if x is not None and not (x.is_cuda and x.dtype == dt and x.is_contiguous() and tuple(x.shape) == shape):
                raise ValueError(f"camera outputs must be contiguous CUDA tensors of shape {shape}")
        _check(lib().mdg_render_depth(self._h, C.byref(c), C.c_void_p(depth.data_ptr() if depth is not None else None),
                                      C.c_void_p(seg.data_ptr() if seg is not None else None)))
        return depth, seg

    def render_rgba(self, cam: mdg_cam_params = None, rgba=None):
        """Every drone's colour frame from the current state (include/mdg.h: mdg_render_rgba): [D, H, W, 4] uint8 CUDA tensor."""
        t = self._torch
        c = cam if cam is not None else default_cam_params(self.params)
        shape = (self.n_envs * self.n_drones, c.height, c.width, 4)
        if rgba is None:
            rgba = t.empty(shape, dtype=t.uint8, device=self.obs.device)
        if not (rgba.is_cuda and rgba.dtype == t.uint8 and rgba.is_contiguous() and tuple(rgba.shape) == shape):
            raise ValueError(f"rgba must be a contiguous CUDA uint8 tensor of shape {shape}")
        _check(lib().mdg_render_rgba(self._h, C.byref(c), C.c_void_p(rgba.data_ptr())))
        return rgba

    def get_state(self):
        import numpy as np
        D = self.n_envs * self.n_drones
        st, ct, tg = np.zeros((D, 13), np.float32), np.zeros((D, 10), np.float32), np.zeros((D, 4), np.float32)
        wd, ep = np.zeros((self.n_envs, 3), np.float32), np.zeros(self.n_envs, np.uint32)
        _check(lib().mdg_get_state(self._h, *[C.c_void_p(a.ctypes.data) for a in (st, ct, tg, wd, ep)]))
        return dict(state=st, ctrl=ct, targets=tg, wind=wd, ep_step=ep)

    def get_dr(self):
        """Domain-randomisation factors of the running episodes, [D, 16] float32 (include/mdg.h: mdg_get_dr)."""
        import numpy as np
        out = np.zeros((self.n_envs * self.n_drones, 16), dtype=np.float32)
        _check(lib().mdg_get_dr(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def set_dr(self, factors):
        import numpy as np
        a = np.ascontiguousarray(factors, dtype=np.float32).reshape(self.n_envs * self.n_drones, 16)
        _check(lib().mdg_set_dr(self._h, a.ctypes.data_as(C.c_void_p)))

    def set_state(self, state=None, ctrl=None, targets=None, wind=None, ep_step=None):
        import numpy as np
        D = self.n_envs * self.n_drones
        spec = ((state, (D, 13), np.float32), (ctrl, (D, 10), np.float32), (targets, (D, 4), np.float32),
                (wind, (self.n_envs, 3), np.float32), (ep_step, (self.n_envs,), np.uint32))
        keep, ptrs = [], []
        for a, shape, dt in spec:
            if a is None:
                ptrs.append(C.c_void_p(None))
            else:
                b = np.ascontiguousarray(a, dtype=dt).reshape(shape)
                keep.append(b)
                ptrs.append(C.c_void_p(b.ctypes.data))
        _check(lib().mdg_set_state(self._h, *ptrs))

    @property
    def launch_count(self):
        return int(lib().mdg_launch_count(self._h))

    @property
    def kernel_name(self):
        return lib().mdg_kernel_name(self._h).decode()

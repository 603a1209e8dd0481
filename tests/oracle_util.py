"""Helpers for the oracle pin tests (CPU only)."""
import os

import numpy as np

from oracle import oracle as O
from paper_2606_08039_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")

FREE = dict(term_mode=W.TERM_NONE, auto_reset=0, episode_len_s=0.0)   # no termination, no reset


def golden_table(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v, tol = line.split()
            out[k] = (float(v), float(tol))
    return out


def make_env(n_envs=1, n_drones=1, physics=W.PHYS_MJC, action=W.ACT_RPM, model=0, threads=1, **over):
    P = O.OracleParams(model, **over)
    env = O.OracleEnv(n_envs, n_drones, physics, action, P, n_threads=threads)
    env.reset(1)
    return env, P


def set_state(env, p=None, q=None, v=None, w=None):
    s = env.state
    D = s.shape[0]
    if p is not None:
        s[:, 0:3] = np.asarray(p, dtype=float).reshape(-1, 3) * np.ones((D, 1))
    if q is not None:
        s[:, 3:7] = np.asarray(q, dtype=float).reshape(-1, 4) * np.ones((D, 1))
    if v is not None:
        s[:, 7:10] = np.asarray(v, dtype=float).reshape(-1, 3) * np.ones((D, 1))
    if w is not None:
        s[:, 10:13] = np.asarray(w, dtype=float).reshape(-1, 3) * np.ones((D, 1))
    env.state = s


def quat_wxyz_from_scipy(r):
    x, y, z, w = r.as_quat()
    return np.array([w, x, y, z])


def scipy_from_wxyz(q):
    from scipy.spatial.transform import Rotation
    return Rotation.from_quat([q[1], q[2], q[3], q[0]])

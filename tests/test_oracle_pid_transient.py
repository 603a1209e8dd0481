"""Pin of the oracle's COUPLED cascaded-PID transient in x / y (Eq.9; small-angle attitude target PAPER.md:353;
Table 6 gains), which the fixed-point and z-axis pins of test_oracle_control_env.py leave open.

For a waypoint a micrometre away the closed loop is linear to O(eps^2): each horizontal axis is the textbook chain
position PID -> tilt target a / g -> attitude PID torque -> double integrator J theta'' = tau -> x'' = g theta, sampled with a
zero-order hold at the control rate.  That chain is iterated here in plain numpy as a 6-state discrete linear system
(nothing of the oracle is called) and compared with the oracle's full nonlinear rigid body.  The loop is isotropic (equal x / y
gains, J_xx = J_yy), so the same scalar response must appear on both world axes at ANY yaw: a wrong sign or a swapped sine /
cosine in the heading rotation or in the roll / pitch targets sends the response the wrong way."""
import math

import numpy as np
import pytest

from oracle_util import FREE, make_env, set_state
from paper_2606_08039_b200 import workloads as W

G, J = 9.81, 1.4e-5                                       # Table 2
KP, KI, KD = 0.4, 0.01, 0.9                               # Table 6, position loop, x / y
KPA, KIA, KDA = 2e-3, 0.0, 5e-4                           # Table 6, attitude loop, roll / pitch
H, K = 1.0 / 240.0, 5
DT = H * K


def unit_step_response(steps):
    """x(t) / eps at the end of every control step for a unit waypoint step, linearised loop, zero initial state."""
    x = vx = th = om = Ix = Ith = 0.0
    out = []
    for _ in range(steps):
        e = 1.0 - x
        Ix += e * DT
        a = KP * e + KI * Ix - KD * vx                     # Eq.9 with v* = 0 (gravity feed-forward cancels the weight)
        e_th = a / G - th                                  # small-angle tilt target
        Ith += e_th * DT
        alpha = (KPA * e_th + KIA * Ith - KDA * om) / J    # held over the K substeps
        for _ in range(K):                                 # wrench from the start-of-substep state, constant over the substep
            x, vx = x + vx * H + 0.5 * G * th * H * H, vx + G * th * H
            th, om = th + om * H + 0.5 * alpha * H * H, om + alpha * H
        out.append(x)
    return np.array(out)


@pytest.mark.parametrize("psi0", [0.0, 0.7, -2.4])
@pytest.mark.parametrize("direction", [(1.0, 0.0), (0.0, 1.0), (-0.6, 0.8)])
def test_small_waypoint_step_follows_the_linearised_cascade_on_both_axes_at_any_yaw(psi0, direction):
    eps = 2.0 ** -20                                       # 0.95 um, exact in fp32
    psi = float(np.float32(psi0))
    env, _ = make_env(action=W.ACT_PID, **FREE)
    set_state(env, p=[0, 0, 1.0], q=[math.cos(psi / 2), 0, 0, math.sin(psi / 2)], v=[0, 0, 0], w=[0, 0, 0])
    a = np.array([[eps * direction[0], eps * direction[1], 1.0, psi]], dtype=np.float32)
    steps = 144                                            # 3 s
    ref = unit_step_response(steps)
    got = np.zeros((steps, 2))
    for t in range(steps):
        env.step(a)
        got[t] = env.state[0, 0:2] / eps
    want = ref[:, None] * np.array(direction, dtype=np.float64)[None, :].astype(np.float32).astype(np.float64)
    assert np.abs(got - want).max() < 2e-5, np.abs(got - want).max()
    assert ref.max() > 0.5 and ref[10] > 1e-4 and np.abs(np.diff(ref)).max() < 0.05      # a real transient, well resolved
    assert abs(env.state[0, 2] - 1.0) < 1e-9               # altitude untouched to first order

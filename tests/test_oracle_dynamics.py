"""Pins of the float64 oracle's dynamics (SURVEY.md §8(c) "Pins"; north_star closed forms).

Every expected value here comes from the paper's equations evaluated by hand (tests/golden/), from a
closed-form solution of the equations of motion, from an invariant, or from a library routine
(scipy Rotation) — never from the oracle itself or from the CUDA path.
"""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import oracle as O
from oracle_util import FREE, golden_table, make_env, quat_wxyz_from_scipy, scipy_from_wxyz, set_state
from paper_2606_08039_b200 import workloads as W

G = golden_table("closed_forms_cf2x.txt")


def _close(val, key):
    ref, tol = G[key]
    assert abs(val - ref) <= tol * abs(ref), (key, val, ref)


# ---- O1 constants (Table 2) --------------------------------------------------------
def test_derived_constants():
    P = O.OracleParams()
    d = P.derived()
    _close(d["hover_rpm"], "hover_rpm")
    _close(d["max_rpm"], "max_rpm")
    _close(d["W"], "W")
    _close(d["W"] / 4, "s_hover")
    _close(d["s_max"], "s_max")
    _close(d["l"], "l")
    _close(d["kappa"], "kappa")
    _close(P.get("h_clip"), "h_clip")
    assert d["K"] == 5 and d["ep_steps"] == 480
    assert abs(d["max_rpm"] / d["hover_rpm"] - 1.5) < 1e-12           # sqrt(2.25)


def test_physics_mode_table1():
    """Table 1: mode -> (aero mask, integrator)."""
    P = O.OracleParams()
    exp = {W.PHYS_MJC: (0, 0), W.PHYS_MJC_GND: (1, 0), W.PHYS_MJC_DRAG: (2, 0), W.PHYS_MJC_DW: (4, 0),
           W.PHYS_MJC_GND_DRAG_DW: (7, 0), W.PHYS_DYN: (0, 1)}
    for mode, (aero, integ) in exp.items():
        d = P.derived(mode)
        assert (d["aero"], d["integ"]) == (aero, integ)
    P["aero_mask"] = 3
    assert P.derived(W.PHYS_MJC)["aero"] == 3                          # params override (config 2)


def test_sim_freq_must_be_multiple_of_ctrl_freq():
    """PAPER.md:169."""
    P = O.OracleParams(sim_freq=250, ctrl_freq=48)
    with pytest.raises(ValueError):
        O.OracleEnv(1, 1, 0, 0, P)


# ---- rotation helpers against scipy (library routine) ---------------------------------------------
def test_euler_and_exp_map_against_scipy():
    rng = np.random.default_rng(0)
    for _ in range(50):
        r = Rotation.random(random_state=rng.integers(1 << 30))
        q = quat_wxyz_from_scipy(r)
        eta = O.euler_zyx(q)
        yaw, pitch, roll = r.as_euler("ZYX")
        assert np.allclose(eta, [roll, pitch, yaw], atol=1e-12)
        phi = rng.normal(size=3) * rng.choice([1e-10, 1e-3, 0.5, 3.0])
        out = O.quat_exp_step(q, phi)                                  # Eq.7: q (x) exp(phi), body-frame phi
        ref = quat_wxyz_from_scipy(r * Rotation.from_rotvec(phi))
        out = out / np.linalg.norm(out)
        assert min(np.abs(out - ref).max(), np.abs(out + ref).max()) < 1e-12


# ---- translation -----------------------------------------------------------------------------------
def test_free_fall_rk4_exact_and_dyn_closed_form():
    """Zero RPM: z(t) = z0 - g t^2 / 2 in MJC mode; DYN: z_n = z0 - g h^2 n (n+1) / 2 (SURVEY pin O4/O8)."""
    g, h = 9.81, 1 / 240
    for phys in (W.PHYS_MJC, W.PHYS_DYN):
        env, _ = make_env(physics=phys, **FREE)
        set_state(env, p=[0.3, -0.2, 100.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        for k in range(1, 49):
            env.step(np.zeros(4))
            n = 5 * k
            z = env.state[0, 2]
            if phys == W.PHYS_MJC:
                ref = 100.0 - 0.5 * g * (n * h) ** 2
            else:
                ref = 100.0 - 0.5 * g * h * h * n * (n + 1)
            assert abs(z - ref) < 1e-11
        s = env.state[0]
        assert abs(s[9] + g * 1.0) < 1e-12 and np.allclose(s[[0, 1]], [0.3, -0.2], atol=1e-15)
        assert np.allclose(s[3:7], [1, 0, 0, 0], atol=1e-15) and np.allclose(s[10:13], 0)
    # the printed DYN number of SURVEY.md: 4.92544 m after 240 substeps vs 4.905 exact
    assert abs(0.5 * g * h * h * 240 * 241 - 4.92544) < 1e-5


def test_hover_equilibrium():
    """All rotors at sqrt(mg/4kf), level, at rest, aero off: nothing moves (north_star)."""
    n = 16384.0                                                        # exactly representable fp32 action
    kf = 0.027 * 9.81 / (4 * n * n)
    for phys in (W.PHYS_MJC, W.PHYS_DYN):
        env, P = make_env(physics=phys, k_f=kf, **FREE)
        assert abs(P.derived()["hover_rpm"] - n) < 1e-9
        set_state(env, p=[0.1, 0.2, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        s0 = env.state.copy()
        for _ in range(48):
            env.step(np.full(4, n))
        assert np.abs(env.state - s0).max() < 1e-12


def test_uniform_thrust_closed_form():
    """Uniform RPM n: z'' = 4 kf n^2 / m - g (Eq.1, T = sum F_i)."""
    env, P = make_env(**FREE)
    n = 15000.0
    acc = 4 * 3.16e-10 * n * n / 0.027 - 9.81
    set_state(env, p=[0, 0, 1.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    for _ in range(48):
        env.step(np.full(4, n))
    s = env.state[0]
    assert abs(s[2] - (1.0 + 0.5 * acc)) < 1e-12 and abs(s[9] - acc) < 1e-12
    assert np.allclose(s[10:13], 0, atol=1e-15)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_pure_axis_torque_closed_form(axis):
    """Eq.1-3 sign patterns: rotor pairs that give a pure roll / pitch / yaw torque with sum F = const.
    Constant torque about a fixed principal axis: w = tau t / J, angle = tau t^2 / (2 J)."""
    a, b = 15000.0, 14000.0
    kf, km, L = 3.16e-10, 7.94e-12, 0.0397
    J = [1.4e-5, 1.4e-5, 2.17e-5]
    if axis == 0:        # tau_x = l (F0 + F1 - F2 - F3)
        rpm = [a, a, b, b]; tau = (L / np.sqrt(2)) * kf * 2 * (a * a - b * b)
    elif axis == 1:      # tau_y = l (-F0 + F1 + F2 - F3)
        rpm = [b, a, a, b]; tau = (L / np.sqrt(2)) * kf * 2 * (a * a - b * b)
    else:                # tau_z = km (-n0^2 + n1^2 - n2^2 + n3^2), reading Q3
        rpm = [b, a, b, a]; tau = km * 2 * (a * a - b * b)
    T, tb, _ = O.motor_wrench(O.OracleParams(), rpm)
    exp_tb = np.zeros(3); exp_tb[axis] = tau
    assert np.allclose(tb, exp_tb, rtol=1e-12, atol=1e-18)
    assert abs(T - kf * 2 * (a * a + b * b)) < 1e-15
    env, _ = make_env(**FREE)
    set_state(env, p=[0, 0, 50.0], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
    t = 0.0
    for _ in range(6):                                                 # 0.125 s
        env.step(rpm)
        t += 1 / 48
        s = env.state[0]
        w_ref = np.zeros(3); w_ref[axis] = tau * t / J[axis]
        assert np.allclose(s[10:13], w_ref, rtol=1e-11, atol=1e-12)
        eta = O.euler_zyx(s[3:7])
        ang = tau * t * t / (2 * J[axis])
        assert abs(eta[axis] - ang) < 1e-10 * max(1, ang)


# ---- torque-free rotation ------------------------------------------------------------------------
def _spin(phys, sim_freq, w0, steps=48):
    env, _ = make_env(physics=phys, sim_freq=sim_freq, **FREE)
    q0 = quat_wxyz_from_scipy(Rotation.from_euler("ZYX", [0.3, -0.2, 0.5]))
    set_state(env, p=[0, 0, 500.0], q=q0, v=[0, 0, 0], w=w0)
    for _ in range(steps):
        env.step(np.zeros(4))
    return q0, env.state[0]


def test_torque_free_rotation_invariants_and_axisymmetric_top():
    """Zero RPM, w0 != 0: |q| = 1, world angular momentum R J w conserved, and for Jxx = Jyy the closed
    form: w_z constant, (w_x, w_y) rotating at (Jzz - Jxx)/Jxx * w_z = 0.55 w_z (SURVEY pin O8)."""
    J = np.array([1.4e-5, 1.4e-5, 2.17e-5])
    w0 = np.array([3.0, -2.0, 100.0])
    lam = (J[2] - J[0]) / J[0] * w0[2]
    assert abs(lam / w0[2] - 0.55) < 1e-12
    errs = {}
    for phys in (W.PHYS_MJC, W.PHYS_DYN):
        # explicit Euler is only in its asymptotic regime for lam*h << 1: use a slower spin there
        w0 = np.array([3.0, -2.0, 100.0]) if phys == W.PHYS_MJC else np.array([3.0, -2.0, 10.0])
        lam = (J[2] - J[0]) / J[0] * w0[2]
        for f in (240, 480):
            q0, s = _spin(phys, f, w0)
            q, w = s[3:7], s[10:13]
            assert abs(np.linalg.norm(q) - 1) < 1e-14
            c, sn = np.cos(lam * 1.0), np.sin(lam * 1.0)
            w_ref = np.array([w0[0] * c - w0[1] * sn, w0[0] * sn + w0[1] * c, w0[2]])
            L0 = scipy_from_wxyz(q0).apply(J * w0)
            L1 = scipy_from_wxyz(q).apply(J * w)
            errs[(phys, f)] = (np.abs(w - w_ref).max(), np.abs(L1 - L0).max() / np.linalg.norm(L0))
            assert abs(w[2] - w0[2]) < 1e-9
    # RK4 is 4th order (error ratio ~16 when h halves), explicit Euler 1st order (~2)
    r_rk4 = errs[(W.PHYS_MJC, 240)][0] / errs[(W.PHYS_MJC, 480)][0]
    r_eul = errs[(W.PHYS_DYN, 240)][0] / errs[(W.PHYS_DYN, 480)][0]
    assert 12 < r_rk4 < 20, r_rk4
    assert 1.7 < r_eul < 2.4, r_eul
    assert errs[(W.PHYS_MJC, 240)][0] < 1e-2 and errs[(W.PHYS_MJC, 240)][1] < 1e-3
    rL = errs[(W.PHYS_MJC, 240)][1] / errs[(W.PHYS_MJC, 480)][1]
    # The body rates converge at 4th order, but the orientation update of reading Q11 (one exponential
    # of the RK4-weighted mean rate from q0, which is also how MuJoCo's RK4 advances a free joint) drops
    # the commutator term, so R J w drifts at O(h^2): ratio ~4, not the 16 SURVEY.md's pin table hoped
    # for (note on Q11).
    assert 3.5 < rL < 4.5, rL


def test_torque_free_orientation_against_closed_form():
    """Axisymmetric free top: body z precesses about the fixed angular momentum at rate |L|/Jxx; the
    oracle's orientation converges to it at 2nd order (see the note in the test above)."""
    J = np.array([1.4e-5, 1.4e-5, 2.17e-5])
    w0 = np.array([3.0, -2.0, 100.0])
    err = {}
    for f in (960, 1920):
        q0, s = _spin(W.PHYS_MJC, f, w0, steps=24)                     # t = 0.5 s
        R0, R1 = scipy_from_wxyz(q0), scipy_from_wxyz(s[3:7])
        Lw = R0.apply(J * w0)
        rate = np.linalg.norm(Lw) / J[0]
        z0, z1 = R0.apply([0, 0, 1.0]), R1.apply([0, 0, 1.0])
        z_ref = Rotation.from_rotvec(Lw / np.linalg.norm(Lw) * rate * 0.5).apply(z0)
        err[f] = np.abs(z1 - z_ref).max()
    assert err[960] < 5e-5 and 3.5 < err[960] / err[1920] < 4.5, err


# ---- aero closed forms (probe the substep wrench) ---------------------------------------------------
def test_ground_effect_closed_forms():
    """Eq.4 at hover RPM, level; clip gain 4/15; zero when inverted."""
    env, P = make_env(physics=W.PHYS_MJC_GND, **FREE)
    n = P.derived()["hover_rpm"]
    T, _, _ = O.motor_wrench(P, [n] * 4)
    for h, key in ((0.05, "gnd_h0.05"), (0.1, "gnd_h0.1"), (1.0, "gnd_h1.0")):
        set_state(env, p=[0, 0, h], q=[1, 0, 0, 0], v=[0, 0, 0], w=[0, 0, 0])
        F, tau = env.probe_wrench(0, [n] * 4)
        _close(F[0, 2] - T, key)
        assert np.allclose(F[0, :2], 0) and np.allclose(tau, 0, atol=1e-18)
    for h in (0.0, 0.01, P.get("h_clip")):
        set_state(env, p=[0, 0, h])
        F, _ = env.probe_wrench(0, [n] * 4)
        _close((F[0, 2] - T) / T, "gnd_gain_clip")
    set_state(env, p=[0, 0, 0.05], q=[0, 1, 0, 0])                     # upside down
    F, _ = env.probe_wrench(0, [n] * 4)
    assert abs(F[0, 2] + T) < 1e-15
    # gate is on the body z axis pointing up: 80 deg roll still gains, 100 deg does not
    for deg, on in ((80, True), (100, False)):
        q = quat_wxyz_from_scipy(Rotation.from_euler("x", deg, degrees=True))
        set_state(env, p=[0, 0, 0.05], q=q)
        F, _ = env.probe_wrench(0, [n] * 4)
        extra = F[0, 2] - T * np.cos(np.radians(deg))
        assert (extra > 1e-3) == on


def test_blade_drag_closed_form_and_equivariance():
    """Eq.5: level, v = x: F = -c_xy * sum(2 pi n / 60) x; general attitude via scipy."""
    env, P = make_env(physics=W.PHYS_MJC_DRAG, **FREE)
    n = P.derived()["hover_rpm"]
    T, _, Om = O.motor_wrench(P, [n] * 4)
    assert abs(Om - 4 * 2 * np.pi * n / 60) < 1e-9
    set_state(env, p=[0, 0, 1], q=[1, 0, 0, 0], v=[1, 0, 0], w=[0, 0, 0])
    F, _ = env.probe_wrench(0, [n] * 4)
    assert np.allclose(F[0], [-9.1785e-7 * Om, 0, T], rtol=1e-12, atol=1e-18)
    set_state(env, v=[0, 0, 1])
    F, _ = env.probe_wrench(0, [n] * 4)
    assert np.allclose(F[0], [0, 0, T - 10.311e-7 * Om], rtol=1e-12, atol=1e-18)
    rng = np.random.default_rng(1)
    c = np.array([9.1785e-7, 9.1785e-7, 10.311e-7])
    for _ in range(20):
        r = Rotation.random(random_state=rng.integers(1 << 30))
        v = rng.normal(size=3)
        rpm = rng.uniform(10000, 20000, size=4)
        T, tb, Om = O.motor_wrench(P, rpm)
        set_state(env, q=quat_wxyz_from_scipy(r), v=v)
        F, tau = env.probe_wrench(0, rpm)
        F_ref = r.apply([0, 0, T]) + r.apply(-c * Om * r.inv().apply(v))
        assert np.allclose(F[0], F_ref, rtol=1e-11, atol=1e-15)
        assert np.allclose(tau[0], r.apply(tb), rtol=1e-11, atol=1e-18)    # PAPER.md:106 world-frame torque
        # yaw-rotation equivariance
        rz = Rotation.from_euler("z", rng.uniform(-3, 3))
        set_state(env, q=quat_wxyz_from_scipy(rz * r), v=rz.apply(v))
        F2, _ = env.probe_wrench(0, rpm)
        assert np.allclose(F2[0], rz.apply(F[0]), rtol=1e-10, atol=1e-15)


def _dw_pair(dz, dxy, **over):
    env, P = make_env(n_drones=2, physics=W.PHYS_MJC_DW, **FREE, **over)
    s = env.state
    s[0, 0:3] = [0.2, -0.1, 1.0]
    s[1, 0:3] = [0.2 + dxy * 0.6, -0.1 + dxy * 0.8, 1.0 + dz]
    env.state = s
    n = P.derived()["hover_rpm"]
    T, _, _ = O.motor_wrench(P, [n] * 4)
    F, _ = env.probe_wrench(0, [[n] * 4, [n] * 4])
    return T - F[0, 2], T - F[1, 2], F


def test_downwash_closed_forms():
    """Eq.6 on the lower of two drones; upper one unaffected (Q10)."""
    for dz, dxy, key in ((0.5, 0.0, "dw_0.5_0"), (1.0, 0.05, "dw_1.0_0.05"), (0.5, 0.1, "dw_0.5_0.1"), (0.1, 0.3, "dw_0.1_0.3")):
        low, up, F = _dw_pair(dz, dxy)
        _close(low, key)
        assert up == 0.0 and np.allclose(F[:, :2], 0)
    low, up, _ = _dw_pair(0.6875, 0.1)                                 # beta = 0: zero off-axis
    assert abs(low) < 1e-300 and up == 0.0
    low, _, _ = _dw_pair(0.5, 10.0)                                    # lateral cut-off
    assert low == 0.0
    # regularisation Q9: below dz_clip the force ramps linearly to zero; dz_clip = 0 is Eq.6 verbatim
    ref, _, _ = _dw_pair(0.1, 0.3)
    half, _, _ = _dw_pair(0.05, 0.3)
    assert abs(half - 0.5 * ref) < 1e-15
    raw, _, _ = _dw_pair(0.05, 0.3, dw_dz_clip=0.0)
    a = 2267.18 * (0.02325 / (4 * 0.05)) ** 2
    b = 0.16 * 0.05 - 0.11
    assert abs(raw - a * np.exp(-0.5 * (0.3 / b) ** 2)) < 1e-12 * raw
    same, _, _ = _dw_pair(0.5, 0.1, dw_dz_clip=0.0)
    _close(same, "dw_0.5_0.1")


def test_downwash_sums_over_all_upper_drones():
    """O(M^2) pair loop: the force on a drone is the sum of the two-drone forces of everyone above it."""
    rng = np.random.default_rng(5)
    M = 5
    env, P = make_env(n_drones=M, physics=W.PHYS_MJC_DW, **FREE)
    s = env.state
    s[:, 0:2] = rng.uniform(-0.2, 0.2, size=(M, 2))
    s[:, 2] = rng.uniform(0.3, 1.5, size=M)
    env.state = s
    n = P.derived()["hover_rpm"]
    T, _, _ = O.motor_wrench(P, [n] * 4)
    F, _ = env.probe_wrench(0, np.full((M, 4), n))
    for i in range(M):
        tot = 0.0
        for k in range(M):
            dz = s[k, 2] - s[i, 2]
            if k == i or dz <= 0:
                continue
            dxy = np.hypot(s[k, 0] - s[i, 0], s[k, 1] - s[i, 1])
            pair, _ = make_env(n_drones=2, physics=W.PHYS_MJC_DW, **FREE)
            ps = pair.state
            ps[0, 0:3] = [0, 0, 1.0]; ps[1, 0:3] = [dxy, 0, 1.0 + dz]
            pair.state = ps
            Fp, _ = pair.probe_wrench(0, np.full((2, 4), n))
            tot += T - Fp[0, 2]
        assert abs((T - F[i, 2]) - tot) < 1e-13


# ---- symmetries ------------------------------------------------------------------------------------
def _random_env(M, seed, **over):
    rng = np.random.default_rng(seed)
    env, P = make_env(n_drones=M, physics=W.PHYS_MJC_GND_DRAG_DW, reward_mode=W.REW_MULTI_HOVER, **FREE, **over)
    s = env.state
    s[:, 0:2] = rng.uniform(-0.3, 0.3, size=(M, 2))
    s[:, 2] = rng.uniform(0.3, 1.2, size=M)
    for i in range(M):
        s[i, 3:7] = quat_wxyz_from_scipy(Rotation.from_rotvec(rng.normal(size=3) * 0.2))
    s[:, 7:10] = rng.normal(size=(M, 3)) * 0.3
    s[:, 10:13] = rng.normal(size=(M, 3)) * 0.5
    tg = env.targets
    tg[:, 0:3] = rng.uniform(-0.3, 0.3, size=(M, 3)) + [0, 0, 1]
    acts = rng.uniform(0.9, 1.1, size=(10, M, 4)) * P.derived()["hover_rpm"]
    return env, s, tg, acts.astype(np.float32)


def test_permutation_symmetry():
    M = 6
    env, s, tg, acts = _random_env(M, 7)
    perm = np.random.default_rng(8).permutation(M)
    env.state = s; env.targets = tg
    env2, _, _, _ = _random_env(M, 7)
    env2.state = s[perm]; env2.targets = tg[perm]
    for a in acts:
        env.step(a)
        env2.step(a[perm])
    assert np.abs(env.state[perm] - env2.state).max() < 1e-12
    o1, r1, _, _ = env.outputs()
    o2, r2, _, _ = env2.outputs()
    assert np.abs(o1.reshape(M, -1)[perm] - o2.reshape(M, -1)).max() < 1e-12 and abs(r1[0] - r2[0]) < 1e-12


def test_translation_and_yaw_rotation_symmetry():
    M = 4
    env, s, tg, acts = _random_env(M, 11)
    env.state = s; env.targets = tg
    for a in acts:
        env.step(a)
    out = env.state
    # translation in x, y
    envT, _, _, _ = _random_env(M, 11)
    sT = s.copy(); sT[:, 0:2] += [0.7, -1.3]
    envT.state = sT
    for a in acts:
        envT.step(a)
    oT = envT.state; oT[:, 0:2] -= [0.7, -1.3]
    assert np.abs(oT - out).max() < 1e-12
    # rotation about z of the initial state rotates the trajectory
    rz = Rotation.from_euler("z", 0.9)
    envR, _, _, _ = _random_env(M, 11)
    sR = s.copy()
    sR[:, 0:3] = rz.apply(s[:, 0:3]); sR[:, 7:10] = rz.apply(s[:, 7:10])
    for i in range(M):
        sR[i, 3:7] = quat_wxyz_from_scipy(rz * scipy_from_wxyz(s[i, 3:7]))
    envR.state = sR
    for a in acts:
        envR.step(a)
    oR = envR.state
    assert np.abs(oR[:, 0:3] - rz.apply(out[:, 0:3])).max() < 1e-12
    assert np.abs(oR[:, 7:10] - rz.apply(out[:, 7:10])).max() < 1e-12
    assert np.abs(oR[:, 10:13] - out[:, 10:13]).max() < 1e-12          # body rates unchanged (Q22)
    for i in range(M):
        qr = quat_wxyz_from_scipy(rz * scipy_from_wxyz(out[i, 3:7]))
        assert min(np.abs(oR[i, 3:7] - qr).max(), np.abs(oR[i, 3:7] + qr).max()) < 1e-12


# ---- floor -----------------------------------------------------------------------------------------
def test_floor_clamp():
    """Q15: p_z < 0 -> p_z = 0, v_z = max(v_z, 0), sticky hit flag -> HOVER termination + crash reward."""
    env, _ = make_env(term_mode=W.TERM_HOVER, auto_reset=0)
    set_state(env, p=[0.4, 0, 0.001], q=[1, 0, 0, 0], v=[0.5, 0, -1.0], w=[0, 0, 0])
    env.step(np.zeros(4))
    s = env.state[0]
    assert s[2] == 0.0 and s[9] == 0.0 and abs(s[7] - 0.5) < 1e-15     # no friction
    _, rew, done, _ = env.outputs()
    assert done[0] == 1 and rew[0] < -100
    # a drone that stays above the floor does not terminate
    set_state(env, p=[0, 0, 1.0], v=[0, 0, 0])
    env.step(np.zeros(4))
    assert env.outputs()[2][0] == 0

"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (sanitizer builds of the native test
infrastructure).  tests/sanitize_oracle_main.cpp links oracle/oracle_capi.cpp into an instrumented executable and runs small
versions of the benchmark workloads through reset / step / auto-reset / camera, on two threads; any out-of-bounds access,
use after free, signed overflow, misaligned access or invalid shift aborts it (-fno-sanitize-recover)."""
import os
import shutil
import subprocess

import pytest

from paper_2606_08039_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def exe(tmp_path_factory):
    if shutil.which("g++") is None:
        pytest.skip("no g++")
    out = str(tmp_path_factory.mktemp("san") / "oracle_san")
    cmd = ["g++", "-std=c++17", "-O1", "-g", "-ffp-contract=off", "-pthread", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-o", out, os.path.join(ROOT, "tests", "sanitize_oracle_main.cpp"), os.path.join(ROOT, "oracle", "oracle_capi.cpp")]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and "sanitize" in r.stderr.lower() and "cannot find" in r.stderr.lower():
        pytest.skip("sanitizer runtime libraries are not installed")
    assert r.returncode == 0, r.stderr[-2000:]
    return out


def scenario(path, wl, n_envs, n_steps, extra=None):
    kind = wl.actions[0]
    base = W.hover_rpm_f32() if kind == "hover_scale" else 1.0
    lo, hi = (wl.actions[1], wl.actions[2]) if kind != "targets" else (-1.0, 1.0)
    lines = [f"{n_envs} {wl.n_drones} {wl.physics_mode} {wl.action_type} {n_steps} {wl.seed} {base!r} {lo} {hi} 2"]
    for k, v in dict(wl.params, **(extra or {})).items():
        for i, x in enumerate(v if isinstance(v, (list, tuple)) else [v]):
            lines.append(f"{k} {i} {float(x)!r}")
    open(path, "w").write("\n".join(lines) + "\n")


@pytest.mark.parametrize("c,variant,n_envs", [(1, None, 1), (2, None, 13), (3, None, 11), (4, None, 5), (5, None, 9), (5, "table4", 9), (5, "dyn", 7)])
def test_oracle_runs_clean_under_asan_and_ubsan(exe, tmp_path, c, variant, n_envs):
    wl = W.config(c)
    extra = dict(W.VARIANTS[variant]) if variant else {}
    extra["episode_len_s"] = 7 / 48                 # auto-resets inside the run
    path = str(tmp_path / "scenario.txt")
    scenario(path, wl, n_envs, 20, extra)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe, path], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, (r.stdout[-500:], r.stderr[-3000:])
    assert r.stdout.startswith("ok ") and "runtime error" not in r.stderr and "Sanitizer" not in r.stderr, r.stderr[-3000:]

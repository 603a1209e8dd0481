"""Build oracle/liboracle.so (TEST INFRASTRUCTURE — the float64 CPU oracle, see drone_oracle.hpp).

Run as `python oracle/build.py`; `__graft_entry__.build()` calls `build()` too.  Plain g++, no CUDA.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "oracle_capi.cpp")]
DEPS = SRC + [os.path.join(HERE, "drone_oracle.hpp"), os.path.join(HERE, "philox_ref.hpp"),
               os.path.join(HERE, "camera_oracle.hpp")]
OUT = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in DEPS):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
           "-Wall", "-Wextra", "-o", OUT] + SRC
    subprocess.run(cmd, check=True, cwd=HERE)
    return OUT


if __name__ == "__main__":
    print(build(force=True))

"""Build paper_2606_08039_b200/libmdg.so in-tree with nvcc for sm_100a (`python -m paper_2606_08039_b200.build`)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libmdg.so")
SOURCES = [os.path.join(CSRC, "mdg.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("mdg_dev.cuh", "mdg_step.cuh", "mdg_kernels.cuh", "mdg_camera.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "mdg.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in DEPS):
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", OUT] + SOURCES + ["-lnvrtc", "-ldl", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
    subprocess.run(cmd, check=True, cwd=CSRC)
    return OUT


if __name__ == "__main__":
    print(build(force=True, verbose=True))

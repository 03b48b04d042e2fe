"""Compile the CUDA library for sm_100a:  python -m paper_1301_3460_b200._build  ->  paper_1301_3460_b200/liblgf.so

The .so is built in-tree (git-ignored, but it travels to the GPU box with the repo snapshot)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "liblgf.so")
SOURCES = [os.path.join(CSRC, "lgf_api.cu")]
STATIC_SOURCE = os.path.join(CSRC, "lgf_static.cu")      # lgf_measure_static: the entry point that allocates nothing
DEPS = SOURCES + [STATIC_SOURCE] + [os.path.join(CSRC, f) for f in ("kernels.cuh", "fft_tile.cuh", "fft_fast.cuh", "fft_tma.cuh", "su3.cuh", "slab.cuh", "lgf_slab.inl")] + [
    os.path.join(os.path.dirname(HERE), "include", "lgf.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "--fmad=true", "-Xptxas", "-v",
]
# lgf_api.cu is compiled twice: fp64 (public lgf_* entry points) and, with -DLGF_F32, fp32 (lgf32_* twins)
OBJECTS = [("lgf_api_f64.o", SOURCES, []), ("lgf_api_f32.o", SOURCES, ["-DLGF_F32"]), ("lgf_static.o", [STATIC_SOURCE], [])]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def have_nvcc() -> bool:
    import shutil
    try:
        n = nvcc()
    except RuntimeError:
        return False
    return bool(shutil.which(n))


def up_to_date() -> bool:
    return os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return OUT
    procs = []
    for obj, src, extra in OBJECTS:
        cmd = [nvcc()] + NVCC_FLAGS + extra + ["-c"] + src + ["-o", os.path.join(HERE, obj)]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)))
    log = ""
    for cmd, p in procs:
        out, err = p.communicate()
        log += "# " + " ".join(cmd) + "\n" + err
        if verbose or p.returncode != 0:
            sys.stderr.write(out + err)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared"] + [os.path.join(HERE, o) for o, _, _ in OBJECTS] + ["-o", OUT]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("link failed: " + " ".join(cmd))
    with open(os.path.join(HERE, "ptxas_info.txt"), "w") as f:
        f.write(log)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

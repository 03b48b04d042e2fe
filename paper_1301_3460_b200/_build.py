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
    """Compile and link liblgf.so unless it is newer than every source.  Safe when several processes arrive at once
    (torchrun ranks, pytest-xdist workers): one of them builds under an exclusive file lock while the others wait and then
    find the library up to date; objects and the library are written under temporary names and moved into place, so no
    process ever loads a half-written file."""
    if not force and up_to_date():
        return OUT
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and up_to_date():       # another process built it while this one waited for the lock
                return OUT
            return _build_locked(verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(verbose: bool) -> str:
    tag = ".tmp%d" % os.getpid()
    procs = []
    for obj, src, extra in OBJECTS:
        cmd = [nvcc()] + NVCC_FLAGS + extra + ["-c"] + src + ["-o", os.path.join(HERE, obj + tag)]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)))
    log = ""
    failed = None
    for cmd, p in procs:
        out, err = p.communicate()
        log += "# " + " ".join(cmd).replace(tag, "") + "\n" + err
        if verbose or p.returncode != 0:
            sys.stderr.write(out + err)
        if p.returncode != 0 and failed is None:
            failed = "nvcc failed: " + " ".join(cmd)
    objs = [os.path.join(HERE, o) for o, _, _ in OBJECTS]
    try:
        if failed:
            raise RuntimeError(failed)
        for o in objs:
            os.replace(o + tag, o)
        cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared"] + objs + ["-o", OUT + tag]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("link failed: " + " ".join(cmd))
        os.replace(OUT + tag, OUT)
    finally:
        for f in [o + tag for o in objs] + [OUT + tag]:
            if os.path.exists(f):
                os.remove(f)
    with open(os.path.join(HERE, "ptxas_info.txt"), "w") as f:
        f.write(log)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

"""Builds libsdm.so (the C-ABI library of include/sdm.h) in-tree with nvcc for sm_100a."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libsdm.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
# per-file flags: the coalescence/move kernel must not contract a*b+c into FMA (see its header)
UNITS = {
    "sdm_api.cu": [],
    "sdm_sort.cu": [],
    "sdm_cond.cu": [],
    "sdm_coal_move.cu": ["-fmad=false"],
    "sdm_diag.cu": ["-fmad=false"],
    "sdm_init.cu": ["-fmad=false"],
    "sdm_recycle.cu": [],
    "sdm_peak.cu": [],
    "sdm_euler.cu": ["-fmad=false"],
    "sdm_slab.cu": [],
    "sdm_noalloc.cu": [],
}
HEADERS = ["sdm_common.cuh", "sdm_kernels.cuh", os.path.join("..", "..", "include", "sdm.h")]


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build(force=False, verbose=False):
    """Compiles csrc/*.cu and links libsdm.so.  SDM_NVCC_EXTRA (environment) appends flags, e.g. -D tuning macros,
    to every unit and forces a rebuild."""
    os.makedirs(OBJ, exist_ok=True)
    env_extra = os.environ.get("SDM_NVCC_EXTRA", "").split()
    force = force or bool(env_extra)
    hdrs = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    objs, jobs = [], []
    for src, extra in UNITS.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + hdrs):
            cmd = [NVCC] + ARCH + COMMON + extra + env_extra + ["-c", s, "-o", o]
            jobs.append((src, o, cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = []
    for src, o, cmd, proc in jobs:   # the translation units compile side by side
        log = proc.communicate()[0]
        with open(o + ".log", "w") as f:
            f.write(" ".join(cmd) + "\n" + log)
        if proc.returncode != 0:
            sys.stderr.write(log)
            failed.append(src)
        elif verbose:
            print(log)
    if failed:
        raise RuntimeError("nvcc failed on " + ", ".join(failed))
    if force or _stale(SO, objs):
        cmd = [NVCC] + ARCH + ["-shared", "-o", SO] + objs
        subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

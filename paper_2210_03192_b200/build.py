"""Builds liblx.so (hand-written CUDA for sm_100a) in-tree with nvcc.  No JIT cache, no torch extension machinery:
the shared library travels with the repository snapshot to the GPU box."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblx.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]

# tuning aid: extra nvcc flags (e.g. "-DLX_TEAM_BUDGET=40") from the environment; they force a rebuild
EXTRA = os.environ.get("LX_EXTRA_NVCC", "").split()
NVCC_FLAGS += EXTRA

LX_RANGE = range(7)      # aux angular momentum 0..LX_MAX_L_AUX
MODES = range(4)         # 0 store, 1 gamma, 2 J, 3 store with solid-harmonic aux functions


def _headers():
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hs.append(os.path.join(os.path.dirname(HERE), "include", "lx.h"))
    return hs


def _units():
    units = [("lx_api.o", "lx_api.cu", [])]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith(".cu") and f not in ("lx_api.cu", "lx_inst.cu"):
            units.append((f[:-3] + ".o", f, []))
    for lx in LX_RANGE:
        for mode in MODES:
            units.append((f"lx_inst_{lx}_{mode}.o", "lx_inst.cu", [f"-DINST_LX={lx}", f"-DINST_MODE={mode}"]))
    return units


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(verbose=False, force=False, jobs=None):
    os.makedirs(OBJ, exist_ok=True)
    hdrs = _headers()
    # objects made with other flags (a tuning build with LX_EXTRA_NVCC) must not be reused: the flags are stamped
    stamp = os.path.join(OBJ, "flags.txt")
    flags_now = " ".join(NVCC_FLAGS)
    if not os.path.exists(stamp) or open(stamp).read() != flags_now:
        force = True
    todo = []
    objs = []
    for obj, src, defs in _units():
        o = os.path.join(OBJ, obj)
        s = os.path.join(CSRC, src)
        objs.append(o)
        if force or _stale(o, [s] + hdrs):
            todo.append(["nvcc"] + NVCC_FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    if todo:
        with ThreadPoolExecutor(max_workers=jobs or os.cpu_count() or 4) as ex:
            for log in ex.map(run, todo):
                if verbose and log:
                    sys.stderr.write(log)
    with open(stamp, "w") as f:
        f.write(flags_now)
    if todo or _stale(LIB, objs):
        run(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(verbose="-v" in sys.argv, force="-f" in sys.argv))

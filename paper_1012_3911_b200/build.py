"""Build libsso.so in-tree with nvcc for sm_100a (no torch extension machinery: the library is plain C ABI).

`python -m paper_1012_3911_b200.build` (or `build()` from Python) compiles
  csrc/sso_api.cu                      the C ABI, plan builder and auxiliary kernels
  csrc/sso_inst.cu  x (precision, N)   the pass kernel, one object per line length and precision
in parallel and links them into paper_1012_3911_b200/libsso.so.  Objects are cached under
paper_1012_3911_b200/build/ and rebuilt when a source or header is newer.

Environment: SSO_SIZES="256,2048" restricts the line lengths that get real kernels (development
only; the other sizes then report SSO_ERR_UNSUPPORTED), SSO_JOBS sets the parallelism, SSO_NVCC_EXTRA adds
nvcc flags to the kernel objects (development, e.g. -DSSO_TIMELINE prints a per-phase clock trace of one group).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "build"
LIB = HERE / "libsso.so"
ALL_SIZES = [16, 32, 64, 128, 256, 512, 1024, 2048, 4096, 8192]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=default",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or Path(cand).exists()):
            return cand
    raise RuntimeError("nvcc not found")


def _newest_source() -> float:
    srcs = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + [HERE.parent / "include" / "sso.h", Path(__file__)]
    return max(p.stat().st_mtime for p in srcs)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: " + " ".join(map(str, cmd)) + "\n" + r.stdout + r.stderr)
    return r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False) -> Path:
    nvcc = _nvcc()
    OBJ.mkdir(exist_ok=True)
    sizes_env = os.environ.get("SSO_SIZES")
    real = set(int(s) for s in sizes_env.split(",")) if sizes_env else set(ALL_SIZES)
    extra = os.environ.get("SSO_NVCC_EXTRA", "").split()  # development: extra nvcc flags (e.g. -DSSO_TIMELINE)
    stamp = _newest_source()
    jobs = []
    objs = []
    api_o = OBJ / "sso_api.o"
    objs.append(api_o)
    if force or not api_o.exists() or api_o.stat().st_mtime < stamp:
        jobs.append([nvcc, *NVCC_FLAGS, "-c", str(CSRC / "sso_api.cu"), "-o", str(api_o)])
    for tname, t in (("f64", "double"), ("f32", "float")):
        for n in ALL_SIZES:
            stub = n not in real
            o = OBJ / f"sso_inst_{tname}_{n}{'_stub' if stub else ''}.o"
            objs.append(o)
            if force or not o.exists() or o.stat().st_mtime < stamp:
                cmd = [nvcc, *NVCC_FLAGS, *extra, f"-DSSO_T={t}", f"-DSSO_TNAME={tname}", f"-DSSO_N={n}"]
                if stub:
                    cmd.append("-DSSO_STUB")
                jobs.append(cmd + ["-c", str(CSRC / "sso_inst.cu"), "-o", str(o)])
    # biggest kernels first so the pool drains evenly
    jobs.sort(key=lambda c: -max([int(x.split("=")[1]) for x in c if x.startswith("-DSSO_N=")] + [10**6 if "sso_api" in " ".join(map(str, c)) else 0]))
    nj = int(os.environ.get("SSO_JOBS", str(os.cpu_count() or 4)))
    if jobs:
        if verbose:
            print(f"[sso build] compiling {len(jobs)} objects with {nj} jobs", file=sys.stderr)
        with ThreadPoolExecutor(max_workers=nj) as ex:
            list(ex.map(_run, jobs))
    if jobs or force or not LIB.exists():
        tmp = LIB.with_suffix(f".so.{os.getpid()}.tmp")
        _run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, objs)])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))

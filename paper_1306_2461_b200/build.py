"""Build liboptflow.so (sm_100a only) in-tree with nvcc.  `python -m paper_1306_2461_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liboptflow.so")
SOURCES = ["optflow.cu", "optflow_hoist.cu", "optflow_hoist_mask.cu", "optflow_mask.cu", "optflow_dual.cu", "optflow_static.cu"]     # compiled in parallel (one nvcc process each), then linked
HEADER = os.path.join("..", "..", "include", "optflow.h")
COMMON = ["of_dispatch.cuh", "of_kernels.cuh", "of_common.cuh", "of_k2.cuh", "of_k2s.cuh", "of_async.cuh", "of_fused.cuh", "of_k3.cuh", "of_solve.cuh",
          "of_equalise.cuh", "of_post.cuh", HEADER]
# what each translation unit includes (an object is recompiled when it is older than its source or one of these)
DEPS = {src: COMMON for src in SOURCES}
DEPS["optflow_dual.cu"] = COMMON + ["of_solve_dual.cuh"]
DEPS["optflow_static.cu"] = [HEADER]
# OF_NVCC_DEFS="--split-compile 8" cuts the build from ~140 s to ~50 s, but nvcc then picks a different register allocation from
# run to run (measured: 156/160, 162/156 or 166/168 registers for the two R = 12 solve kernels), so it is not the default:
# the library that is tested must be the library that is rebuilt from the same sources.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _obj(src: str) -> str:
    return os.path.join(HERE, "build", os.path.splitext(src)[0] + ".o")


def _stale_sources(flags_line: str) -> list:
    """Translation units whose object is missing, older than the source or a header it includes, or built with other flags."""
    stamp = os.path.join(HERE, "build", "flags.txt")
    if not os.path.exists(stamp) or open(stamp).read() != flags_line:
        return list(SOURCES)
    out = []
    for src in SOURCES:
        o = _obj(src)
        if not os.path.exists(o):
            out.append(src)
            continue
        t = os.path.getmtime(o)
        if any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in [src] + DEPS[src]):
            out.append(src)
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    defs = os.environ.get("OF_NVCC_DEFS", "").split()
    flags_line = " ".join([nvcc] + NVCC_FLAGS + defs)
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    todo = list(SOURCES) if force else _stale_sources(flags_line)
    if todo or not os.path.exists(LIB):
        tmp = LIB + ".tmp.%d" % os.getpid()
        objs = [_obj(src) for src in SOURCES]
        cmds = [[nvcc] + NVCC_FLAGS + defs + ["-c", "-o", _obj(src), os.path.join(CSRC, src)] for src in todo]
        procs = [subprocess.Popen(c, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for c in cmds]
        outs = [pr.communicate()[0] for pr in procs]
        rc = max([pr.returncode for pr in procs] + [0])
        link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs
        if rc == 0:
            r = subprocess.run(link, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
            outs.append(r.stdout)
            rc = r.returncode
        log = "".join(" ".join(c) + "\n" + o for c, o in zip(cmds + [link], outs))
        with open(os.path.join(HERE, "build.log"), "a" if (todo != list(SOURCES)) else "w") as f:
            f.write(log)
        if verbose or rc != 0:
            sys.stderr.write(log)
        if rc != 0:
            for src, pr in zip(todo, procs):                      # a failed unit must be compiled again next time
                if pr.returncode != 0 and os.path.exists(_obj(src)):
                    os.remove(_obj(src))
            raise RuntimeError("nvcc failed (see %s)" % os.path.join(HERE, "build.log"))
        with open(os.path.join(HERE, "build", "flags.txt"), "w") as f:
            f.write(flags_line)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))

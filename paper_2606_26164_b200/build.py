"""Build libchisao.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a:  python -m paper_2606_26164_b200.build

nvcc cross-compiles without a GPU.  The five objective instantiations are separate translation units and
are compiled in parallel.  The resulting paper_2606_26164_b200/libchisao.so is git-ignored but travels to
the GPU box with the repository snapshot.
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libchisao.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]
if os.environ.get("CHISAO_EXPERIMENTS"):      # ablation switches of the tensor-core kernels (profiles/; selected by CHISAO_EXP at run time)
    FLAGS.append("-DCHISAO_EXPERIMENTS")

UNITS = [("chisao_api.cu", []), ("chisao_lbfgs.cu", []), ("chisao_select.cu", []), ("chisao_tc_kernels.cu", []), ("chisao_stencil.cu", []), ("chisao_probe.cu", []), ("chisao_static.cu", [])] + \
        [("chisao_eval_obj.cu", [f"-DCHISAO_OBJ_INST={i}"]) for i in range(6)]


def _headers():
    hs = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h"))]
    hs.append(os.path.join(os.path.dirname(HERE), "include", "chisao.h"))
    return hs


def _stamp(src, extra):
    h = hashlib.sha256()
    for p in [src] + _headers():
        with open(p, "rb") as f:
            h.update(f.read())
    h.update(" ".join(FLAGS + extra).encode())
    return h.hexdigest()


def _compile(unit):
    name, extra = unit
    src = os.path.join(CSRC, name)
    tag = name.replace(".cu", "") + ("_" + extra[0].split("=")[1] if extra else "")
    obj = os.path.join(OBJDIR, tag + ".o")
    stamp_file = obj + ".stamp"
    stamp = _stamp(src, extra)
    if os.path.exists(obj) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return obj, False
    cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
    subprocess.check_call(cmd)
    with open(stamp_file, "w") as f:
        f.write(stamp)
    return obj, True


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJDIR, exist_ok=True)
    if force:
        for f in os.listdir(OBJDIR):
            os.remove(os.path.join(OBJDIR, f))
    with cf.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        res = list(ex.map(_compile, UNITS))
    objs = [o for o, _ in res]
    if any(changed for _, changed in res) or not os.path.exists(LIB):
        cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"]
        subprocess.check_call(cmd)
        if verbose:
            print("linked", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))

"""Builds the native libraries in-tree (no JIT cache): datagen (C), encoder (C++) and the CUDA decoder (sm_100a).  `python -m paper_2606_18900_b200.build [target...]`."""
import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)

CUDA_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--use_fast_math",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _newer(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd, log=None):
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if log:
        with open(log, "w") as f:
            # without the "Compile time" lines the log is the same for the same source
            f.write(" ".join(cmd) + "\n" + "".join(ln for ln in r.stdout.splitlines(True) if "Compile time" not in ln))
    if r.returncode != 0:
        raise RuntimeError("build failed: %s\n%s" % (" ".join(cmd), r.stdout))
    return r.stdout


def build_datagen(force=False):
    src = [os.path.join(PKG, "datagen", "datagen.c")]
    out = os.path.join(PKG, "datagen", "libacx_datagen.so")
    if force or _newer(out, src):
        _run(["gcc", "-O2", "-Wall", "-shared", "-fPIC", "-o", out] + src)
    return out


def build_encoder(force=False):
    src = [os.path.join(PKG, "encoder", "encoder.cpp")]
    out = os.path.join(PKG, "encoder", "libacx_encoder.so")
    if force or _newer(out, src):
        _run(["g++", "-O2", "-std=c++17", "-Wall", "-shared", "-fPIC", "-pthread", "-o", out] + src)
    return out


def build_cuda(force=False):
    cs = os.path.join(PKG, "csrc")
    src = [os.path.join(cs, f) for f in sorted(os.listdir(cs)) if f.endswith(".cu")]
    deps = src + [os.path.join(cs, f) for f in os.listdir(cs) if f.endswith((".cuh", ".h"))]
    deps.append(os.path.join(ROOT, "include", "aceapex.h"))
    out = os.path.join(PKG, "libaceapex.so")
    if force or _newer(out, deps):
        nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
        _run([nvcc] + CUDA_FLAGS + ["-I", os.path.join(ROOT, "include"), "-o", out] + src + ["-lcudart"],
             log=os.path.join(PKG, "ptxas_v.log"))          # build log: registers, spills, shared memory (git-ignored)
    return out


TARGETS = {"datagen": build_datagen, "encoder": build_encoder, "cuda": build_cuda}


def build_all(force=False):
    return {k: f(force) for k, f in TARGETS.items()}


if __name__ == "__main__":
    names = [a for a in sys.argv[1:] if not a.startswith("-")] or list(TARGETS)
    for n in names:
        print(n, "->", TARGETS[n]("--force" in sys.argv))

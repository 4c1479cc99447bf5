"""TEST INFRASTRUCTURE ONLY.  Compiles the product's .cu sources as plain C++ (g++) against the fiber-based CUDA
emulation in this directory -> tests/cuda_emul/libnrr_bm_emul.so.  The CPU tests use it to run the kernels' logic
without a GPU; the product package never loads it."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2308_10868_b200", "csrc")
SOURCES = ["nrr_api.cu", "nrr_select.cu", "nrr_boxstat.cu", "nrr_match.cu", "nrr_match_pair.cu", "nrr_plan.cu", "nrr_fem.cu", "nrr_warp.cu"]   # not the FFMA microbenchmark
ASAN = os.environ.get("NRR_EMUL_ASAN", "0") == "1"      # AddressSanitizer build: LD_PRELOAD libasan when loading it
LIB = os.path.join(HERE, "libnrr_bm_emul_asan.so" if ASAN else "libnrr_bm_emul.so")
FLAGS = ["-std=c++17", "-O1", "-g", "-ffp-contract=off", "-fPIC", "-fvisibility=hidden", "-fno-strict-aliasing",
         "-Wno-attributes", "-Wno-unknown-pragmas", "-I", os.path.join(HERE, "include")]
if ASAN:
    # alignment: a misaligned float4 / double2 / ulonglong2 access (a misaligned-address fault on the GPU) aborts here
    FLAGS += ["-fsanitize=address", "-fsanitize=alignment", "-fno-sanitize-recover=alignment", "-fno-omit-frame-pointer"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "nrr_bm.h")]
    deps += [os.path.join(HERE, "emul.cpp"), os.path.join(HERE, "stubs.cpp"), os.path.abspath(__file__)]
    deps += [os.path.join(HERE, "include", f) for f in os.listdir(os.path.join(HERE, "include"))]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    objdir = os.path.join(HERE, "build", "asan" if ASAN else "plain")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        procs.append((src, subprocess.Popen(["g++", "-x", "c++"] + FLAGS + ["-c", os.path.join(CSRC, src), "-o", obj],
                                            stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src in ("emul.cpp", "stubs.cpp"):
        obj = os.path.join(objdir, src.replace(".cpp", ".o"))
        procs.append((src, subprocess.Popen(["g++"] + FLAGS + ["-c", os.path.join(HERE, src), "-o", obj],
                                            stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            sys.stderr.write("---- %s\n%s\n" % (src, out))
            failed = True
    if failed:
        raise RuntimeError("g++ failed building the CUDA emulation")
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["g++", "-shared"] + (["-fsanitize=address", "-fsanitize=alignment"] if ASAN else []) + ["-o", tmp] + objs, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

"""Build libfdas_emu.so: the product's CUDA sources (paper_1511_07343_b200/csrc) compiled as host C++
against the shim in this folder.  TEST INFRASTRUCTURE ONLY -- see README.md here."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_1511_07343_b200", "csrc")
OUT = os.path.join(HERE, "build")
LIB = os.path.join(OUT, "libfdas_emu.so")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps += [os.path.join(HERE, f) for f in ("cuda_runtime.h", "emu_tma.h", "emu_rt.cpp", "selftest_tma.cpp", "prep.py", "build.py")]
    deps.append(os.path.join(ROOT, "include", "fdas.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    try:
        from . import prep
    except ImportError:                                  # run as a script
        import prep
    src_dir = os.path.join(OUT, "pkg", "csrc")          # mirrors <pkg>/csrc so "../../include/fdas.h" resolves
    os.makedirs(src_dir, exist_ok=True)
    os.makedirs(os.path.join(OUT, "include"), exist_ok=True)
    shutil.copy(os.path.join(ROOT, "include", "fdas.h"), os.path.join(OUT, "include", "fdas.h"))
    units = []
    for f in sorted(os.listdir(CSRC)):
        if f == "fdas_tma.cuh":                          # inline PTX: emu_tma.h stands in for it (prep.py)
            continue
        text = prep.rewrite(open(os.path.join(CSRC, f)).read())
        dst = os.path.join(src_dir, f[:-3] + ".cpp" if f.endswith(".cu") else f)
        open(dst, "w").write(text)
        if f.endswith(".cu"):
            units.append(dst)
    units.append(os.path.join(HERE, "emu_rt.cpp"))
    units.append(os.path.join(HERE, "selftest_tma.cpp"))
    procs, objs = [], []
    for u in units:
        o = os.path.join(OUT, os.path.basename(u)[:-4] + ".o")
        objs.append(o)
        cmd = ["g++", "-std=c++17", "-O2", "-g", "-fPIC", "-fno-strict-aliasing", "-fsanitize=alignment",
               "-fno-sanitize-recover=alignment", "-I", HERE, "-c", u, "-o", o]
        procs.append((u, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for u, p in procs:
        out, _ = p.communicate()
        if p.returncode:
            raise RuntimeError("g++ failed on %s:\n%s" % (u, out))
    subprocess.check_call(["g++", "-shared", "-fsanitize=alignment", "-o", LIB, *objs, "-lpthread"])
    return LIB


if __name__ == "__main__":
    print(build(force=True))

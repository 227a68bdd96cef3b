"""Build libopd.so (csrc/opd_lib.cu) for sm_100a with nvcc, in-tree.

    python -m paper_2606_24143_b200.build [--force] [--verbose]
    python -m paper_2606_24143_b200.build --sass-histogram      # tcgen05 / TMEM / TMA opcodes per kernel of the built library
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libopd.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    raise RuntimeError("nvcc not found")


def sources():
    out = [os.path.join(INCLUDE, "opd.h")]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".inl")):
            out.append(os.path.join(CSRC, f))
    return out


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC", "-I", INCLUDE,
           os.path.join(CSRC, "opd_lib.cu"), "-o", LIB]
    cmd[1:1] = os.environ.get("OPD_NVCC_FLAGS", "").split()
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libopd.so")
    return LIB


def sass_histogram() -> str:
    """Per kernel of the built libopd.so: how many tensor-core (UTC*MMA = tcgen05.mma), TMEM (LDTM / STTM = tcgen05.ld / st),
    TMA (UTMALDG / UTMASTG / UTMAREDG = cp.async.bulk.tensor loads, stores, reductions) and tcgen05 barrier / allocation
    (UTCBAR, UTCATOMSWS) instructions its SASS holds; HMMA (mma.sync) would show a legacy tensor-core path."""
    import collections
    import re
    sass = subprocess.run(["cuobjdump", "-sass", build()], capture_output=True, text=True, check=True).stdout
    pat = re.compile(r"\b(UTC\w*MMA[.\w]*|UTMA\w+[.\w]*|LDTM[.\w]*|STTM[.\w]*|UTCBAR[.\w]*|UTCCP[.\w]*|UTCATOM\w*[.\w]*|HMMA[.\w]*|UBLKCP[.\w]*)")
    per_fn, fn = collections.OrderedDict(), None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            per_fn.setdefault(fn, collections.Counter())
        elif fn is not None:
            m = pat.search(line)
            if m:
                per_fn[fn][m.group(1)] += 1
    out = []
    for fn, cnt in per_fn.items():
        if not cnt:
            continue
        name = subprocess.run(["c++filt", fn], capture_output=True, text=True).stdout.strip() or fn
        out.append(re.sub(r"\(CUtensorMap_st.*", "(...)", name))
        out += [f"    {v:6d}  {k}" for k, v in sorted(cnt.items())]
    return "\n".join(out) + "\n"


if __name__ == "__main__":
    if "--sass-histogram" in sys.argv:
        sys.stdout.write(sass_histogram())
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))

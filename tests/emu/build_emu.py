"""Build tests/emu/libgsr_emu.so: the kernels and the C ABI of paper_2503_22863_b200/csrc compiled for the HOST
against tests/emu/cuda_runtime.h (one OS thread per CUDA thread).  TEST INFRASTRUCTURE ONLY -- see the header of
tests/emu/cuda_runtime.h.  The .cu sources are used as they are, except for the two things g++ cannot parse:

  kernel<<<grid, block, smem, stream>>>(args);   ->  emu::launch(grid, block, smem, stream, [=] { kernel(args); });
  extern __shared__ char smem_raw[];             ->  (the global smem_raw of the emulator)

GSR_EMU_SANITIZE=address|thread|undefined builds an instrumented variant (libgsr_emu_<san>.so).
"""
import glob
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2503_22863_b200", "csrc")
GEN = os.path.join(HERE, "_gen")


def so_path(sanitize: str = "") -> str:
    return os.path.join(HERE, "libgsr_emu" + (f"_{sanitize}" if sanitize else "") + ".so")


def _balanced(text: str, i: int) -> int:
    """text[i] == '(' -> index one past the matching ')'."""
    depth = 0
    for j in range(i, len(text)):
        c = text[j]
        if c == "(":
            depth += 1
        elif c == ")":
            depth -= 1
            if depth == 0:
                return j + 1
    raise ValueError("unbalanced parentheses in a kernel launch")


def _split_args(s: str):
    out, depth, cur = [], 0, ""
    for c in s:
        if c in "([{":
            depth += 1
        elif c in ")]}":
            depth -= 1
        if c == "," and depth == 0:
            out.append(cur.strip())
            cur = ""
        else:
            cur += c
    out.append(cur.strip())
    return out


def rewrite(src: str) -> str:
    src = src.replace("extern __shared__ char smem_raw[];", "/* dynamic shared memory: the emulator's global smem_raw */")
    out, pos = "", 0
    for m in re.finditer(r"([A-Za-z_][A-Za-z0-9_]*)\s*<<<", src):
        if m.start() < pos:
            continue
        end_cfg = src.index(">>>", m.end())
        cfg = _split_args(src[m.end():end_cfg])
        cfg += ["0", "nullptr"][len(cfg) - 2:] if len(cfg) < 4 else []
        open_paren = end_cfg + 3
        while src[open_paren].isspace():
            open_paren += 1
        assert src[open_paren] == "(", "kernel launch without an argument list"
        close = _balanced(src, open_paren)
        args = src[open_paren + 1:close - 1]
        semi = close
        while src[semi].isspace():
            semi += 1
        assert src[semi] == ";", "kernel launch is not a statement"
        out += src[pos:m.start()]
        out += (f"emu::launch({cfg[0]}, {cfg[1]}, {cfg[2]}, {cfg[3]}, [=] {{ {m.group(1)}({args}); }});")
        pos = semi + 1
    return out + src[pos:]


def build(force: bool = False, sanitize: str = None) -> str:
    sanitize = os.environ.get("GSR_EMU_SANITIZE", "") if sanitize is None else sanitize
    so = so_path(sanitize)
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    deps = srcs + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(HERE, "*.h")) + \
        glob.glob(os.path.join(HERE, "*.cpp")) + [os.path.join(ROOT, "include", "gsr.h"), os.path.abspath(__file__)]
    if not force and os.path.exists(so) and all(os.path.getmtime(d) <= os.path.getmtime(so) for d in deps):
        return so
    os.makedirs(GEN, exist_ok=True)
    gen = []
    for p in srcs:
        q = os.path.join(GEN, os.path.basename(p)[:-3] + ".emu.cpp")
        with open(p) as f, open(q, "w") as g:
            g.write(f'#line 1 "{p}"\n' + rewrite(f.read()))
        gen.append(q)
    cmd = [os.environ.get("GSR_EMU_CXX", "g++"), "-std=c++20", "-O1", "-g", "-fPIC", "-shared", "-pthread", "-mfma",
           "-ffp-contract=off", "-DGSR_HOST_EMULATION", "-Wall", "-Wno-unknown-pragmas", "-Wno-unused-function",
           "-Wno-unused-variable", "-Wno-sign-compare", "-Wno-psabi", "-I", HERE, "-I", os.path.join(ROOT, "include"), "-I", CSRC]
    if sanitize:
        cmd += [f"-fsanitize={sanitize}", "-fno-omit-frame-pointer"]
    tmp = so + ".tmp%d" % os.getpid()
    cmd += ["-o", tmp] + gen + [os.path.join(HERE, "emu_runtime.cpp")]
    subprocess.check_call(cmd)
    os.replace(tmp, so)
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

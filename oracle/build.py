"""Build oracle/liboracle.so from oracle/tpc_oracle.cpp (plain g++, no CUDA, no product code)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tpc_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")

# -ffp-contract=off: one rounding per written operation; never -ffast-math.
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall", "-Wextra"]


def _host_flags() -> list[str]:
    """std::fma compiles to one hardware instruction where the host has FMA3, else glibc's
    correctly rounded software fmaf/fma is called: the same bits either way, only the oracle's speed differs."""
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.startswith("flags"):
                    return ["-mfma"] if " fma " in ln + " " else []
    except OSError:
        pass
    return []


def build(force: bool = False) -> str:
    flags = _host_flags()
    stamp = LIB + ".flags"                      # the library travels between hosts: rebuild if it was made for another one
    same_host = os.path.exists(stamp) and open(stamp).read().split() == flags
    if not force and same_host and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["g++", *FLAGS, *flags, SRC, "-o", tmp], check=True)
    os.replace(tmp, LIB)
    with open(stamp, "w") as f:
        f.write(" ".join(flags))
    return LIB


if __name__ == "__main__":
    print(build(force=True))

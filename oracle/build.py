"""Compile oracle/rt_oracle.cpp into oracle/librt_oracle.so (g++, no CUDA)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "rt_oracle.cpp")
OUT = os.path.join(HERE, "librt_oracle.so")


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            return " fma " in f.read()
    except OSError:
        return False


def build(force: bool = False) -> str:
    if (not force and os.path.exists(OUT)
            and os.path.getmtime(OUT) >= os.path.getmtime(SRC)):
        return OUT
    # -ffp-contract=off: no implicit fused multiply-add; the algorithm writes fma explicitly.
    # -mfma only makes std::fma one instruction instead of a libm call (same result).
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
           "-pthread", SRC, "-o", OUT]
    if _cpu_has_fma():
        cmd.insert(1, "-mfma")
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

"""Build the CPU oracle (oracle/feds_oracle.c, feds_oracle_strong.c, feds_oracle_packed.c, feds_oracle_tiled.c) into oracle/libfeds_oracle.so with gcc.

TEST INFRASTRUCTURE. `python -m oracle.build` or `oracle.build.build()`; called by tests/conftest.py,
`__graft_entry__.build()` and bench.py's cpu_baseline leg. Plain `gcc -O2`, no SIMD flags, libm only.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "feds_oracle.c"), os.path.join(HERE, "feds_oracle_strong.c"), os.path.join(HERE, "feds_oracle_packed.c"), os.path.join(HERE, "feds_oracle_tiled.c")]
LIB = os.path.join(HERE, "libfeds_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(f) for f in SRCS):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp] + SRCS + ["-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))

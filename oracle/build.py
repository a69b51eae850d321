"""ORACLE — test infrastructure only.  Compiles oracle/*.hpp + oracle_capi.cpp into liboracle.so
with plain g++ (-O2, no fast-math, so FP64 results follow the written order of operations)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SRCS = ["oracle_capi.cpp"]
DEPS = SRCS + ["common.hpp", "philox.hpp", "rambo.hpp", "dirac.hpp", "me_eemumu.hpp", "me_qcd.hpp", "me_qq.hpp"]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(os.path.join(HERE, f)) for f in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-pthread", "-ffp-contract=off",
           "-o", LIB] + [os.path.join(HERE, s) for s in SRCS]
    subprocess.check_call(cmd, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))

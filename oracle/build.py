"""ORACLE -- TEST INFRASTRUCTURE ONLY.  Compiles oracle/*.cpp into oracle/liboracle.so (g++ -O2)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["rng.cpp", "geometry.cpp", "field.cpp", "physics.cpp", "stepper.cpp", "tables.cpp"]
LIB = os.path.join(HERE, "liboracle.so")


def build(force=False):
    srcs = [os.path.join(HERE, s) for s in SOURCES]
    deps = srcs + [os.path.join(HERE, "oracle.h"), os.path.join(HERE, "internal.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    # -ffp-contract=off: plain IEEE double operations, no fused multiply-add
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-Wall", "-Wextra",
           "-o", LIB] + srcs
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))

"""ORACLE — TEST INFRASTRUCTURE ONLY.  Compiles oracle/*.cpp into oracle/liboracle.so with g++.

Building the checker is not using it: `__graft_entry__.build()` calls this; the product
package never imports anything from here.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SOURCES = ["lincheck.cpp", "mutex_queue.cpp", "apps_cpu.cpp", "oracle_capi.cpp"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for f in os.listdir(HERE):
        if f.endswith((".cpp", ".hpp")) and os.path.getmtime(os.path.join(HERE, f)) > t:
            return True
    return False


def build(force: bool = False) -> str:
    if not force and not _stale():
        return LIB
    srcs = [os.path.join(HERE, s) for s in SOURCES if os.path.exists(os.path.join(HERE, s))]
    # -ffp-contract=off: the CPU ray tracer must round every operation (NEXT-2)
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-pthread", "-ffp-contract=off",
           "-Wall", "-o", LIB] + srcs
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))

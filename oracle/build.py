"""Build the CPU oracle (plain C, gcc) into oracle/libea_oracle.so.

TEST INFRASTRUCTURE: building the checker is not using it.  Called by
`__graft_entry__.build()`, by tests/conftest.py, and by `python -m oracle.build`.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ea_oracle.c")
LIB = os.path.join(HERE, "libea_oracle.so")


def build(force: bool = False) -> str:
    # tests/test_oracle_mutants.py points the loader at a deliberately broken build to show that the pins catch it
    override = os.environ.get("EA_ORACLE_LIB")
    if override:
        return override
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)  # atomic: concurrent test workers never see a half-written file
    return LIB


if __name__ == "__main__":
    print(build(force=True))

"""Build oracle/libsg_oracle.so (gcc, OpenMP).  TEST INFRASTRUCTURE -- see sg_oracle.c."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sg_oracle.c")
LIB = os.path.join(HERE, "libsg_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    objs = []
    for tag, defs in (("f80", []), ("f64", ["-DSG_ORACLE_DOUBLE"])):
        obj = os.path.join(HERE, f"sg_oracle_{tag}.o")
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-fopenmp", "-std=c11", "-fno-fast-math",
                               *defs, "-c", SRC, "-o", obj])
        objs.append(obj)
    subprocess.check_call(["gcc", "-shared", "-fopenmp", "-o", LIB, *objs, "-lm"])
    return LIB


if __name__ == "__main__":
    print(build(force=True))

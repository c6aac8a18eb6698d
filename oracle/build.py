"""Compile oracle/lv_oracle.c into oracle/liblv_oracle.so (TEST INFRASTRUCTURE).

gcc only; -ffp-contract=off so the fp32 contract expressions are evaluated as
written.  Run as `python -m oracle.build` or through `oracle.build.build()`.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lv_oracle.c")
LIB = os.path.join(HERE, "liblv_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


def build_sanitized(out_path: str) -> str:
    """The same source with AddressSanitizer + UndefinedBehaviorSanitizer, for
    tests/test_oracle_sanitize.py; loaded through LV_ORACLE_LIB under LD_PRELOAD=libasan."""
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", out_path, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return out_path


if __name__ == "__main__":
    print(build(force=True))

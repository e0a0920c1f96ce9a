"""Builds oracle/libnecsim_oracle.so (TEST INFRASTRUCTURE). Usage: python oracle/build.py"""
import os, subprocess, sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "necsim_oracle.c")
OUT = os.path.join(HERE, "libnecsim_oracle.so")

def build(force=False):
    deps = [SRC, os.path.join(HERE, "neglog_table.inc")]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall", "-Wextra",
           SRC, "-o", OUT, "-lm"]
    subprocess.check_call(cmd)
    return OUT

if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

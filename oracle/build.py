"""Builds liboracle.so from oracle/*.c with gcc (test infrastructure, see rt_oracle.c header)."""
import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ORACLE_SO = os.path.join(HERE, "liboracle.so")


def build_oracle(force=False):
    src = sorted(glob.glob(os.path.join(HERE, "*.c")))
    if force or not os.path.exists(ORACLE_SO) or any(os.path.getmtime(s) > os.path.getmtime(ORACLE_SO) for s in src):
        # -ffp-contract=off: the oracle's arithmetic is the formula as written, no FMA contraction
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-o", ORACLE_SO, *src, "-lm"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("oracle build failed:\n" + r.stdout + r.stderr)
    return ORACLE_SO


if __name__ == "__main__":
    print(build_oracle(force=True))

"""Build the CPU oracle (test infrastructure) into two shared libraries, one per precision.

    python oracle/build.py

No FMA contraction (-ffp-contract=off): the oracle evaluates every expression exactly as written.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sft_oracle.c")


def lib_path(fp32: bool) -> str:
    return os.path.join(HERE, "libsft_oracle_f32.so" if fp32 else "libsft_oracle_f64.so")


def build(force: bool = False) -> None:
    for fp32 in (False, True):
        out = lib_path(fp32)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
            continue
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c99",
               "-Wall", "-Wextra", "-Wno-unused-parameter"]
        if fp32:
            cmd.append("-DORACLE_FP32")
        cmd += ["-o", out + ".tmp", SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print("built", lib_path(False), lib_path(True))

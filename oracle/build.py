"""Builds oracle/libgenga_oracle.so from the plain-C oracles (kick + pre-check; Rcrit / HC / FG; detection; grouping; Bulirsch-Stoer) (test infrastructure; gcc only)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "genga_kick_oracle.c"), os.path.join(HERE, "genga_step_oracle.c"),
        os.path.join(HERE, "genga_group_oracle.c"), os.path.join(HERE, "genga_bs_oracle.c"),
        os.path.join(HERE, "genga_detect_oracle.c")]
LIB = os.path.join(HERE, "libgenga_oracle.so")
# -ffp-contract=off: every product and sum rounds separately, as the header promises.
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(s) for s in SRCS):
        subprocess.check_call(["gcc", *CFLAGS, *SRCS, "-o", LIB, "-lm"])
    return LIB


if __name__ == "__main__":
    print(build(force=True))

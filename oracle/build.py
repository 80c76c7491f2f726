"""Compile the oracle (su3_oracle.c) into libsu3oracle.so.  Standalone on purpose:
the oracle shares nothing with the CUDA library, not even a build helper."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "su3_oracle.c")
LIB = os.path.join(HERE, "libsu3oracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]
# The same source under AddressSanitizer + UndefinedBehaviorSanitizer: out-of-bounds indexing,
# signed overflow in the index maps, misaligned or invalid loads abort the process instead of going unnoticed.
# tests/test_oracle_sanitized.py runs the pins against this build in a child process (libasan preloaded).
LIB_SAN = os.path.join(HERE, "libsu3oracle_san.so")
CFLAGS_SAN = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
              "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build_sanitized(force: bool = False) -> str:
    if force or not os.path.exists(LIB_SAN) or os.path.getmtime(LIB_SAN) < os.path.getmtime(SRC):
        tmp = LIB_SAN + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc"] + CFLAGS_SAN + ["-o", tmp, SRC])
        os.replace(tmp, LIB_SAN)
    return LIB_SAN


def build(force: bool = False) -> str:
    if os.environ.get("SU3_ORACLE_SANITIZED") == "1":     # set by the sanitizer test for its child process only
        return build_sanitized(force)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc"] + CFLAGS + ["-o", tmp, SRC])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))

"""Build the CPU oracle shared library (oracle/libhzo.so).  Test infrastructure only.

Run as `python oracle/build.py`; `__graft_entry__.build()` calls `build()` too (building the
checker is not using it).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hzo.cpp")
LIB = os.path.join(HERE, "libhzo.so")
FLAGS = ["-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-Wall", "-Wextra"]


SAN_LIB = os.path.join(HERE, "libhzo_san.so")
SAN_FLAGS = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]


def build(force: bool = False, sanitize: bool = False) -> str:
    """sanitize=True builds oracle/libhzo_san.so with AddressSanitizer and UndefinedBehaviorSanitizer (SURVEY.md
    section 5).  The pins run on it with
        HZO_LIB=oracle/libhzo_san.so LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
            python -m pytest tests -m "not gpu" -k oracle
    (oracle/binding.py loads the library HZO_LIB names)."""
    deps = [SRC, os.path.join(HERE, "hzo.h")]
    lib = SAN_LIB if sanitize else LIB
    if (not force) and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps):
        return lib
    flags = [f for f in FLAGS if f != "-O2"] + SAN_FLAGS if sanitize else FLAGS
    cmd = ["g++"] + flags + ["-o", lib, SRC]
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, sanitize="--sanitize" in sys.argv))

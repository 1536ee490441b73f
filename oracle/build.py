"""Builds the CPU oracle (test infrastructure) into oracle/liblbmref.so with g++."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lbmref.cpp")
LIB = os.path.join(HERE, "liblbmref.so")


def build(force=False):
    """ORACLE_SANITIZE=1 in the environment builds oracle/liblbmref_san.so with
    -fsanitize=address,undefined instead; run the pins under it with
        ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) \
            ASAN_OPTIONS=detect_leaks=0 python -m pytest tests -m "not gpu" -k oracle
    (the oracle is test infrastructure: the switch selects which build of the checker the tests load)."""
    if os.environ.get("ORACLE_SANITIZE"):
        lib = os.path.join(HERE, "liblbmref_san.so")
        if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(SRC):
            subprocess.check_call(["g++", "-O1", "-g", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
                                   "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                                   "-fno-omit-frame-pointer", "-Wall", "-Wextra", SRC, "-o", lib])
        return lib
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC),
                                             os.path.getmtime(os.path.join(HERE, "lbmref.h")))):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           SRC, "-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))

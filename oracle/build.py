"""Build the CPU oracle shared library (test infrastructure, see tbsma_oracle.c header).

Usage: python oracle/build.py   ->  oracle/liboracle_tbsma.so
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tbsma_oracle.c")
LIB = os.path.join(HERE, "liboracle_tbsma.so")


SAN_LIB = os.path.join(HERE, "liboracle_tbsma_san.so")


def build(force: bool = False) -> str:
    """ORACLE_SANITIZE=1 in the environment builds (and makes oracle/__init__.py load) the same source under
    AddressSanitizer + UndefinedBehaviorSanitizer; run the pins under it with
        ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
            python -m pytest tests/test_oracle_pins.py -q
    (the preload because the interpreter itself is not instrumented; leak detection off because CPython never frees
    everything at exit).  UBSan is built to abort on the first report, so a finding fails the run."""
    san = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
    lib = SAN_LIB if san else LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    opt = (["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
           if san else ["-O2"])
    cmd = ["gcc"] + opt + ["-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-o", lib, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

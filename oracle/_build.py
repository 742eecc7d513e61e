"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.  One compile step for the three C oracles.

    gcc -O2 -fopenmp -fcx-limited-range -shared -fPIC            (no -ffast-math)

CCSD_ORACLE_SANITIZE=1 builds `<name>_asan.so` with -fsanitize=address,undefined instead (the CPU pins are then run
under LD_PRELOAD=$(gcc -print-file-name=libasan.so); profiles/r02_sanitizers.md records such a run).
"""
import os
import subprocess

SANITIZE = os.environ.get("CCSD_ORACLE_SANITIZE") == "1"


def lib_path(path: str) -> str:
    return path[:-3] + "_asan.so" if SANITIZE else path


def compile_oracle(src: str, lib: str, force: bool = False) -> str:
    lib = lib_path(lib)
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        flags = ["-O2", "-fopenmp", "-fcx-limited-range"]
        if SANITIZE:
            flags = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fopenmp", "-fcx-limited-range"]
        subprocess.check_call(["gcc"] + flags + ["-shared", "-fPIC", "-o", lib, src])
    return lib

"""Build the CPU oracle's C sources into oracle/_oracle.so with gcc.

ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).
Run: python -m oracle.build
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["linattn_oracle.c", "capsule_oracle.c", "gdn_oracle.c"]
TARGET = os.path.join(HERE, "_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(TARGET):
        return True
    t = os.path.getmtime(TARGET)
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in SOURCES)


def build(force: bool = False) -> str:
    if not force and not needs_build():
        return TARGET
    tmp = TARGET + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
           "-o", tmp] + [os.path.join(HERE, s) for s in SOURCES] + ["-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, TARGET)
    return TARGET


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

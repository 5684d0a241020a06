"""Builds oracle/libspiir_oracle.so from spiir_oracle.c with gcc (test infrastructure).

Two builds of the SAME source, neither tuned:
  * the checker (default): -O2, portable, what tests/ and smoke() compare against;
  * the timed build (`timed=True`): -O3 -march=native, as BASELINE.md section 3 states for the CPU
    baseline.  -march=native is only valid on the machine that compiles it, so this one is built
    at run time, on the box bench.py runs on, into a file named after that box's CPU.
Both keep -ffp-contract=off (no fused multiply-adds), so the float32 decision path of O4 rounds
exactly as written in either.
"""
import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "spiir_oracle.c")
LIB = os.path.join(HERE, "libspiir_oracle.so")


def _cpu_tag():
    try:
        txt = open("/proc/cpuinfo").read()
        key = "".join(l for l in txt.splitlines() if l.startswith(("model name", "flags")))[:20000]
    except OSError:
        key = "unknown"
    return hashlib.md5(key.encode()).hexdigest()[:10]


def build(force=False, timed=False):
    lib = os.path.join(HERE, "libspiir_oracle_timed_%s.so" % _cpu_tag()) if timed else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(SRC):
        return lib
    opt = ["-O3", "-march=native"] if timed else ["-O2"]
    cmd = ["gcc"] + opt + ["-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                           "-fvisibility=hidden", "-o", lib, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return lib


def physical_cores():
    """Physical cores of this box (distinct (core, socket) pairs of `lscpu -p`), else the CPU count."""
    try:
        out = subprocess.run(["lscpu", "-p=core,socket"], capture_output=True, text=True, check=True).stdout
        pairs = {l.strip() for l in out.splitlines() if l and not l.startswith("#")}
        if pairs:
            return len(pairs)
    except Exception:
        pass
    return os.cpu_count() or 1


if __name__ == "__main__":
    print(build(force=True))

"""Build the CPU oracle shared library (test infrastructure). `python -m oracle.build`.

Flags: -O3 -march=native with OpenMP over events, as BASELINE.md section 2 states for the timed CPU baseline;
-ffp-contract=off keeps every operation individually rounded (no fused multiply-add), so the oracle's arithmetic does
not depend on the host's instruction set. The library is rebuilt whenever the source, the flags or the host CPU's
feature set change (a -march=native binary built in one container must not be run on another machine).
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "trex_oracle.cpp")
LIB = os.path.join(HERE, "libtrex_oracle.so")
STAMP = LIB + ".stamp"
CMD = ["g++", "-std=c++17", "-O3", "-march=native", "-ffp-contract=off", "-fcx-limited-range", "-fopenmp", "-shared", "-fPIC",
       SRC, "-o", LIB]


def _host_tag():
    flags = ""
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(SRC, "rb") as fh:
        src = fh.read()
    return hashlib.sha256(flags.encode() + b"\0" + " ".join(CMD[:-3]).encode() + b"\0" + src).hexdigest()


def build(force=False):
    tag = _host_tag()
    if not force and os.path.exists(LIB) and os.path.exists(STAMP):
        with open(STAMP) as fh:
            if fh.read().strip() == tag:
                return LIB
    subprocess.check_call(CMD)
    with open(STAMP, "w") as fh:
        fh.write(tag + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))

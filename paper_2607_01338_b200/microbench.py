"""Builds and runs csrc/pipe_microbench.cu on the current GPU and prints its JSON line.

    python -m paper_2607_01338_b200.microbench [--out FILE]

The result (warp instructions per clock per SM of the FP32 / MUFU / ALU / shuffle / shared-memory pipes) is
the measured denominator of the LOS transfer kernel's "alu" roofline.
"""
import json
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "pipe_microbench.cu")
EXE = os.path.join(HERE, "pipe_microbench")


def build():
    if os.path.exists(EXE) and os.path.getmtime(EXE) >= os.path.getmtime(SRC):
        return EXE
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-cudart", "static",
                    "-o", EXE, SRC], check=True)
    return EXE


def sm_clock_mhz():
    try:
        out = subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                             capture_output=True, text=True, check=True).stdout
        return float(out.strip().splitlines()[0])
    except Exception:
        return 1965.0


def run():
    exe = build()
    out = subprocess.run([exe, "%.0f" % sm_clock_mhz()], capture_output=True, text=True, check=True).stdout
    return json.loads(out)


if __name__ == "__main__":
    res = run()
    text = json.dumps(res, indent=1)
    if "--out" in sys.argv:
        with open(sys.argv[sys.argv.index("--out") + 1], "w") as f:
            f.write(text + "\n")
    print(text)

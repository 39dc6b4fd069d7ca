"""Builds the probes with nvcc (sm_100a) into a temporary directory, runs them on cuda:0 and prints their tables.

    python -m paper_2606_21023_b200.probes > gpurun_out/probes.md

They are stand-alone CUDA programs (they only share the inline-PTX header of the library) and measure what bounds the
kernels: the TMA streaming rate from HBM, the floor of a dependent 33.5 MB launch, and the L2 -> SM delivery rate with
and without TMA multicast.
"""
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    with tempfile.TemporaryDirectory() as tmp:
        for name, title in (("tma_stream", "TMA streaming from HBM (tile = 64 k x 128 columns of a 4096-column FP16 matrix)"),
                            ("mc_delivery", "L2 -> SM delivery, unicast vs TMA multicast (32 MB, L2-resident)")):
            exe = os.path.join(tmp, name)
            subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-o", exe,
                                   os.path.join(HERE, name + ".cu"), "-lcuda"])
            out = subprocess.run([exe], capture_output=True, text=True, timeout=600)
            print(f"## {title}\n\n```\n{out.stdout.strip()}\n```\n")
            if out.returncode != 0:
                print(out.stderr[-2000:], file=sys.stderr)
                raise SystemExit(out.returncode)


if __name__ == "__main__":
    main()

"""Build and run probes/pipe_probe.cu (developer tool; needs a B200): issue cost of the instructions of the softmax
loops and of the forward kernel's row step on one SM sub-partition.

    python -m paper_2606_03681_b200.pipe_probe

The binary goes to a temporary directory; nothing of it is part of libtabattn.so.
"""
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))


def compile_probe(out_dir):
    """nvcc probes/pipe_probe.cu for sm_100a into ``out_dir``; returns the path of the binary."""
    src = os.path.join(HERE, "probes", "pipe_probe.cu")
    exe = os.path.join(out_dir, "pipe_probe")
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
                    "-o", exe, src], check=True)
    return exe


def main():
    with tempfile.TemporaryDirectory() as tmp:
        return subprocess.run([compile_probe(tmp)]).returncode


if __name__ == "__main__":
    sys.exit(main())

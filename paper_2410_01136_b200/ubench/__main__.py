"""Microbenchmarks behind the roofline denominators: python -m paper_2410_01136_b200.ubench

  pipes.cu         FFMA / DFMA / MUFU / F2F throughput and dependent-issue latency (the "alu" peak, the FP64 and XU
                   pipe rates the float64 Faraday chain is measured against)
  grid_streams.cu  gather and red.global.add ceilings on config 3's actual index stream (gridded path)

Each is compiled with nvcc for sm_100a into a temporary binary and run on the current GPU."""
import subprocess
import sys
import tempfile
from pathlib import Path

HERE = Path(__file__).resolve().parent


def run(name: str) -> str:
    """Compile <name>.cu for sm_100a into a temporary binary, run it on the current GPU, return its stdout."""
    with tempfile.TemporaryDirectory() as d:
        exe = Path(d) / name
        subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
                        "-o", str(exe), str(HERE / f"{name}.cu")], check=True)
        return subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout


def main():
    which = sys.argv[1:] or ["pipes", "grid_streams"]
    for name in which:
        print(f"== {name}", flush=True)
        print(run(name), end="", flush=True)


if __name__ == "__main__":
    main()

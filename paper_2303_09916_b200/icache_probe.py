"""Instruction-cache probe for sm_100a (the measurement behind the design of csrc/jit_score.cu, profiles/r2b.md).

Generates kernels whose loop body is S independent FFMAs of straight-line code (16 bytes each), compiles them with nvcc
for sm_100a and times them at 4 and 8 resident warps per SM:

    python -m paper_2303_09916_b200.icache_probe --build     # CPU box: writes icache_probe.bin next to this file (minutes)
    python -m paper_2303_09916_b200.icache_probe             # GPU box: runs it and prints one line per (size, occupancy)

Result on B200 (profiles/r2b_icache.txt): full issue rate up to 32 KB of code, ~3 cycles per instruction per warp from
48 KB to 128 KB, ~6 cycles per instruction per warp above 128 KB.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
BIN = os.path.join(HERE, "icache_probe.bin")
SIZES = [1024, 2048, 3072, 4096, 6144, 8192, 9216, 12288]


def source() -> str:
    out = ["#include <cstdio>\n#include <cuda_runtime.h>\n"]
    for S in SIZES:
        out.append(f"__global__ void __launch_bounds__(128) k{S}(float *o, int reps, float s)\n{{\n"
                   "    float a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;\n"
                   "    #pragma unroll 1\n    for (int r = 0; r < reps; ++r) {\n")
        for i in range(S // 8):
            c = 1.0 + 1e-6 * (i % 977)
            out.append("        " + " ".join(f"a{k} = fmaf(a{k}, s, {c}f);" for k in range(8)) + "\n")
        out.append("    }\n    o[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;\n}\n")
    out.append("int main()\n{\n    float *o; cudaMalloc(&o, 148 * 8 * 128 * 4 * 4);\n    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b); float ms;\n"
               "    int clk = 0; cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0); const double hz = clk * 1e3;\n"
               "    printf(\"SM clock used for the cycle counts: %.0f MHz\\n\", hz / 1e6);\n")
    for S in SIZES:
        for blocks in (148 * 2, 148):
            reps = max(1, (1 << 22) // S)
            w = blocks // 148 * 4
            out.append(f"    k{S}<<<{blocks}, 128>>>(o, 2, 0.999f); cudaDeviceSynchronize(); cudaEventRecord(a); k{S}<<<{blocks}, 128>>>(o, {reps}, 0.999f); "
                       "cudaEventRecord(b); cudaEventSynchronize(b); cudaEventElapsedTime(&ms, a, b);\n")
            out.append(f"    printf(\"body %6d instructions (%4d KB)  {w} warps/SM: %.2f cycles per instruction per warp, IPC/SM %.2f\\n\", {S}, {S} * 16 / 1024, "
                       f"ms * 1e-3 * hz / ((double){S} * {reps}), (double){S} * {reps} * {w} / (ms * 1e-3 * hz));\n")
    out.append("    return 0;\n}\n")
    return "".join(out)


def build() -> str:
    src = os.path.join(HERE, "build", "icache_probe.cu")
    os.makedirs(os.path.dirname(src), exist_ok=True)
    with open(src, "w") as f:
        f.write(source())
    subprocess.run([os.environ.get("NVCC", "nvcc"), "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-o", BIN, src], check=True)
    return BIN


if __name__ == "__main__":
    if "--build" in sys.argv:
        print(build())
    else:
        if not os.path.exists(BIN):
            raise SystemExit("run with --build first (cross-compiles without a GPU)")
        sys.exit(subprocess.run([BIN]).returncode)

"""Measures the fp64 no-return atomic-add (RED.ADD.F64) peak of the box for the tally sizes of the
five configs and prints a markdown table.  Measurement support beside bench.py: the
micro-benchmark kernel lives in bench_atomic_peak.cu, outside the product library.

    python bench_atomic_peak.py > profiles/atomic_peak_r2.md
"""
import ctypes as C
import os
import subprocess

ROOT = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(ROOT, "bench_atomic_peak.cu")
LIB = os.path.join(ROOT, "libbench_atomic_peak.so")

SIZES = [("config 1/3 hot bin (1 bin, same address)", 1),
         ("config 3 (20 bins)", 20),
         ("config 2 (200 x 100 bins, 160 KB)", 20_000),
         ("config 4 (51 x 51 x 7 x 10 bins, 1.46 MB)", 182_070),
         ("config 5 hot time slice (64^3 x 7 bins, 14.7 MB)", 1_835_008),
         ("config 5 whole tally (294 MB)", 36_700_160)]


def build(force=False):
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-Xcompiler", "-fPIC",
                        "-shared", "-o", LIB + ".tmp", SRC], check=True)
        os.replace(LIB + ".tmp", LIB)
    return LIB


def main():
    import torch
    L = C.CDLL(build())
    L.bench_atomic_peak.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_int, C.c_void_p, C.POINTER(C.c_double)]
    s = torch.cuda.current_stream()
    print("# fp64 atomic-add peak (RED.ADD.F64, pseudo-random addresses), measured on this box\n")
    print("Command: `python bench_atomic_peak.py`  (", torch.cuda.get_device_name(0), ")\n")
    print("| array | bins | atomics/s | GB/s of 8-byte payload |\n|---|---|---|---|")
    for name, n in SIZES:
        for leader in (0, 1):
            if leader and n > 1000:
                continue          # (large arrays: lanes of a warp seldom share a bin, nothing is aggregated)
            arr = torch.zeros(n, dtype=torch.float64, device="cuda")
            n_ops = 1 << 28 if n > 1000 else (1 << 29 if leader else 1 << 24)
            ms = C.c_double()
            rc = L.bench_atomic_peak(C.c_void_p(arr.data_ptr()), n, n_ops, leader, C.c_void_p(s.cuda_stream), C.byref(ms))
            done = (n_ops + n_ops // 8) // (32 if leader else 1)
            assert rc == 0 and abs(arr.sum().item() - done) < 0.5 + 1e-9 * done
            rate = (n_ops // (32 if leader else 1)) / (ms.value * 1e-3)
            print(f"| {name}{', one lane per warp (aggregated tally)' if leader else ''} | {n} | {rate:.3e} | {rate * 8 / 1e9:.1f} |")


if __name__ == "__main__":
    main()

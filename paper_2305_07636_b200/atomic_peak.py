"""Measures the fp64 no-return atomic-add (RED.ADD.F64) peak of the box for the tally sizes of the
five configs and prints a markdown table.

    python -m paper_2305_07636_b200.atomic_peak > profiles/atomic_peak_r1.md
"""
import ctypes as C

import torch

from .binding import load_library

SIZES = [("config 1/3 hot bin (1 bin, same address)", 1),
         ("config 3 (20 bins)", 20),
         ("config 2 (200 x 100 bins, 160 KB)", 20_000),
         ("config 4 (51 x 51 x 7 x 10 bins, 1.46 MB)", 182_070),
         ("config 5 hot time slice (64^3 x 7 bins, 14.7 MB)", 1_835_008),
         ("config 5 whole tally (294 MB)", 36_700_160)]


def main():
    L = load_library()
    s = torch.cuda.current_stream()
    print("# fp64 atomic-add peak (RED.ADD.F64, pseudo-random addresses), measured on this box\n")
    print("Command: `python -m paper_2305_07636_b200.atomic_peak`  (", torch.cuda.get_device_name(0), ")\n")
    print("| array | bins | atomics/s | GB/s of 8-byte payload |\n|---|---|---|---|")
    for name, n in SIZES:
        arr = torch.zeros(n, dtype=torch.float64, device="cuda")
        n_ops = 1 << 28 if n > 1000 else 1 << 24
        ms = C.c_double()
        rc = L.mcdc_atomic_peak(C.c_void_p(arr.data_ptr()), n, n_ops, C.c_void_p(s.cuda_stream), C.byref(ms))
        assert rc == 0 and abs(arr.sum().item() - (n_ops + n_ops // 8)) < 0.5
        rate = n_ops / (ms.value * 1e-3)
        print(f"| {name} | {n} | {rate:.3e} | {rate * 8 / 1e9:.1f} |")


if __name__ == "__main__":
    main()

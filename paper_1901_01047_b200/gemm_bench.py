"""Micro-benchmark of the library's FP64 DMMA GEMM kernels (ctaux_dgemm_ex) on the shapes of the walker's
GEMM steps, beside cuBLAS (torch) on the same shapes.  CUDA events, 3 warm-up + `reps` timed launches.

    python -m paper_1901_01047_b200.gemm_bench            # table on stdout (markdown)

Kernels (include/ctaux.h): 0 = 128x64 tiles, 8 warps, 2 CTAs/SM; 1 = 64x64, 8 warps; 2/3 = persistent 16-warp
kernel (128x64 / 64x128); 4/5 = same with k-step 32; 6 = 64x64, 4 warps, 4 CTAs/SM; 7 = same at 5 CTAs/SM;
8 = kernel 6 + L2 prefetch of the next-wave C0 tile.  Measurement helper: no CT-AUX arithmetic here."""
from __future__ import annotations

import sys


def _time(fn, reps):
    import torch
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def main():
    import torch
    from . import colmajor, ctaux_dgemm, probe_fp64
    if not torch.cuda.is_available():
        raise SystemExit("no CUDA device")
    print(f"FP64 issue-rate peaks: DMMA.8x8x4 {probe_fp64(0):.1f} TFLOP/s, DFMA {probe_fp64(1):.1f} TFLOP/s\n")
    shapes = [("4096^3, C = A B", 4096, 4096, 4096, 1.0, 0.0, 5),
              ("7336^2 rank 64, C = C - A B (16 flushes of config 4)", 7336, 7336, 64, -1.0, 1.0, 20),
              ("7336^2 rank 128, C = C - A B", 7336, 7336, 128, -1.0, 1.0, 20),
              ("7592 x 256 x 1898 (candidate columns)", 7592, 256, 1898, 1.0, 0.0, 20),
              ("256 x 7336 x 1834 (candidate rows)", 256, 7336, 1834, 1.0, 0.0, 20)]
    kernels = [0, 1, 2, 3, 4, 5, 6, 7, 8]
    g = torch.Generator(device="cpu").manual_seed(1)
    rnd = lambda r, c: torch.randn(r, c, generator=g, dtype=torch.float64)
    print("| shape | " + " | ".join(f"kernel {k}" for k in kernels) + " | cuBLAS (torch) |")
    print("|---|" + "---|" * (len(kernels) + 1))
    for name, M, N, K, al, be, reps in shapes:
        A, B, Cm = colmajor(M, K, fill=rnd), colmajor(K, N, fill=rnd), colmajor(M, N, fill=rnd)
        row = []
        for k in kernels:
            ms = _time(lambda: ctaux_dgemm(A, B, Cm, alpha=al, beta=be, kernel=k), reps)
            row.append(2.0 * M * N * K / ms / 1e9)
        At, Bt, Ct = A.contiguous(), B.contiguous(), Cm.contiguous()
        if be == 0.0:
            ms = _time(lambda: torch.matmul(At, Bt, out=Ct), reps)
        else:
            ms = _time(lambda: Ct.addmm_(At, Bt, alpha=al, beta=be), reps)
        print(f"| {name} | " + " | ".join(f"{v:.1f}" for v in row) + f" | {2.0 * M * N * K / ms / 1e9:.1f} |")
        sys.stdout.flush()


if __name__ == "__main__":
    main()

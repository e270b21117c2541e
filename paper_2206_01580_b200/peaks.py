"""Measures the roofline denominators MEASURED_PEAKS.json does not carry on the current
GPU and prints them as one JSON object:

    python -m paper_2206_01580_b200.peaks > profiles/peaks_r2.json

  * plain-ALU issue rates through libqmll.so's `qmll_microbench` (register-only loops on every SM): FADD, FADD2
    (add.f32x2), FFMA, FFMA2, LOP3, SHF, the sign-flip + butterfly mixes of the SORF kernels, MUFU.COS, SHFL, and the
    shared-memory LDS.128 bandwidth -- each as lane-operations per second (CUDA events, the figure the rooflines use)
    and per clock64 tick and SM (on this part clock64 advances at about half the SM clock, so that column is only
    good for ratios between kinds);
  * the TF32 tensor-core GEMM rate (torch.matmul with TF32 allowed, 8192^3): best of 10 (burst) and back to back for
    4 s (sustained), the method MEASURED_PEAKS.json states for its bf16 figure.
"""
from __future__ import annotations

import ctypes
import json
import sys
import time

import torch

from . import load_library

KINDS = {0: "fadd", 1: "ffma", 2: "fadd2", 3: "ffma2", 4: "lop3", 5: "shf", 6: "fadd2+lop3 (1:1), fp32 adds",
         7: "7 fadd + shf + lop3 (round-1 chain), fp32 adds", 8: "3 fadd2 + fadd + shf + lop3 (packed chain), fp32 adds",
         9: "mufu.cos", 10: "lds.128 bytes", 11: "shfl", 12: "2 fadd2 + shf + lop3, fp32 adds",
         13: "dfma (FP64 FMAs)", 14: "dmma m8n8k4 (FP64 FMAs)"}


def microbench(kind: int, iters: int = 4096, blocks_per_sm: int = 4, reps: int = 5) -> dict:
    lib = load_library()
    lib.qmll_microbench.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t,
                                    ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int), ctypes.c_void_p]
    lib.qmll_microbench.restype = ctypes.c_int
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    ws = torch.zeros(n_sm * blocks_per_sm * (256 * 4 + 8) + 4096, dtype=torch.uint8, device="cuda")
    ops, nb = ctypes.c_double(0.0), ctypes.c_int(0)
    stream = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)

    def run():
        rc = lib.qmll_microbench(kind, iters, blocks_per_sm, ctypes.c_void_p(ws.data_ptr()), ws.numel(),
                                 ctypes.byref(ops), ctypes.byref(nb), stream)
        if rc != 0:
            raise RuntimeError(f"qmll_microbench({kind}) -> {rc}")

    run()
    torch.cuda.synchronize()
    best_ms, cyc = None, None
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        run()
        b.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b)
        if best_ms is None or ms < best_ms:
            best_ms = ms
            cyc = ws[: nb.value * 8].view(torch.int64).double().median().item()
    per_block = ops.value / nb.value
    per_clk_sm = per_block * blocks_per_sm / cyc          # all blocks of an SM are co-resident (4 x 256 threads)
    per_s = ops.value / (best_ms * 1e-3)
    return {"what": KINDS[kind], "per_s": per_s, "per_sm_per_clock_at_1965mhz": per_s / n_sm / 1.965e9,
            "per_clock64_tick_per_sm": per_clk_sm, "ms": best_ms}


def tf32_gemm(n: int = 8192, sustained_s: float = 4.0) -> dict:
    torch.backends.cuda.matmul.allow_tf32 = True
    a = torch.randn(n, n, device="cuda")
    b = torch.randn(n, n, device="cuda")
    c = torch.empty(n, n, device="cuda")
    flops = 2.0 * n ** 3
    for _ in range(3):
        torch.matmul(a, b, out=c)
    torch.cuda.synchronize()
    best = 1e9
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b, out=c)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0, k = time.perf_counter(), 0
    e0.record()
    while time.perf_counter() - t0 < sustained_s:
        for _ in range(10):
            torch.matmul(a, b, out=c)
        k += 10
        torch.cuda.synchronize()
    e1.record()
    torch.cuda.synchronize()
    sus = e0.elapsed_time(e1) / k
    torch.backends.cuda.matmul.allow_tf32 = False
    return {"tf32_tflops_burst": flops / (best * 1e-3) / 1e12, "tf32_tflops_sustained": flops / (sus * 1e-3) / 1e12,
            "how": f"torch.matmul fp32 with allow_tf32, {n}^3: best of 10 (burst) and back to back for {sustained_s} s"}


def mma_clocks(iters: int = 512) -> dict:
    """Clocks per tcgen05.mma (M 128, kind::f16, operands in shared memory) for several widths and accumulator counts."""
    lib = load_library()
    lib.qmll_microbench_mma.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t,
                                        ctypes.c_void_p]
    lib.qmll_microbench_mma.restype = ctypes.c_int
    ws = torch.zeros(1, dtype=torch.int64, device="cuda")
    stream = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    out = {}
    for n, accs in ((64, (1, 2, 4)), (96, (1, 2, 4)), (128, (1, 2, 4)), (256, (1, 2))):
        for r in accs:
            for _ in range(2):
                rc = lib.qmll_microbench_mma(n, r, iters, ctypes.c_void_p(ws.data_ptr()), 8, stream)
                if rc != 0:
                    raise RuntimeError(f"qmll_microbench_mma({n}, {r}) -> {rc}")
                torch.cuda.synchronize()
            out[f"N{n}_acc{r}"] = {"clocks_per_mma": ws.item() / (iters * 4.0 * r), "work_clocks": n / 2}
    out["how"] = "clock64 ticks of one CTA per SM issuing back to back; work_clocks = 128 * N / 256 (tensor-core floor)"
    return out


def main() -> None:
    props = torch.cuda.get_device_properties(0)
    out = {"gpu_name": props.name, "sm_count": props.multi_processor_count, "torch": torch.__version__,
           "when": time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime()),
           "command": "python -m paper_2206_01580_b200.peaks", "alu": {}}
    for k in sorted(KINDS):
        out["alu"][str(k)] = microbench(k)
    out["tensor"] = tf32_gemm()
    out["mma_clocks"] = mma_clocks()
    json.dump(out, sys.stdout, indent=1)
    print()


if __name__ == "__main__":
    main()

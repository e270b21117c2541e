"""bench.py -- one "step" = one pass of the whole SORF hot path over one
batch of synthetic input shaped like BASELINE.json:configs[1] (MD-trajectory-like: 1000 x 21 atoms, d = 128,
D = 8192, E+F training rows + E+F prediction):
    qmll_sorf_forward (+G)  ->  qmll_normal_equations on [Z; G]  ->  qmll_predict (E + F)
Prints ONE JSON line (contract in the task statement; extra keys: roofline, cpu_baseline, e2e, clocks).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n-mol M] [--D D]
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "SORF molecules/s (energy+forces), ZtZ TFLOPS, % of HBM/tensor roofline"
UNIT = "molecules/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c2")
    ap.add_argument("--n-mol", type=int, default=None, help="shrink the workload (debug only; invalid as a bench)")
    ap.add_argument("--D", type=int, default=None, help="shrink the workload (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--report-configs", action="store_true",
                    help="time every call of all five BASELINE.json configs (one JSON line per config); not the bench line")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": p["hbm_gbs"], "bf16_burst": p["bf16_tflops"], "bf16_sustained": p["bf16_tflops_sustained"],
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


# ------------------------------------------------------------------------------------------------ oracle arm
def oracle_sample_step(w):
    """The whole path on workload w with the FP64 oracle as it stands (never tuned)."""
    import numpy as np
    import oracle
    Z = oracle.forward_w(w)
    G = oracle.force_rows_w(w)
    A = np.concatenate([Z, G]).astype(np.float32)
    oracle.normal_equations(A, w.y)
    oracle.predict_w(w)


def time_oracle(cfg, D, sample_mol, steps, warmup):
    import oracle
    from workloads import make_workload
    w = make_workload(cfg, n_mol=sample_mol, D=D)
    oracle.build()
    for _ in range(warmup):
        oracle_sample_step(w)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_sample_step(w)
    dt = (time.perf_counter() - t0) / steps
    return dt, oracle.num_threads(), w


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sample_mol = 2
    full_D = args.D or 8192
    dt, cores, w = time_oracle(args.config, full_D, sample_mol, args.steps, min(args.warmup, 1))
    val = sample_mol / dt
    sample = (f"{sample_mol} of 1000 molecules of {args.config} at full D={full_D}: forward + force rows + FP64 A^T A "
              f"on its {w.n_mol + 3 * w.n_atoms} rows + predict E+F, per step")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "c2: 1000 x C9H8O4 (21 atoms), d=128, D=8192, T=3, dense gradient; oracle on a sample",
                       "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        rows = [r.strip().split(",") for r in self.f.read().strip().splitlines() if r.strip()]
        self.f.close()
        os.unlink(self.f.name)
        sm, reasons, mx, pw = [], set(), None, []
        for r in rows:
            try:
                sm.append(float(r[0])); mx = float(r[1]); pw.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(name)
        if sm:
            sm.sort()
            out.update({"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": mx, "reasons": sorted(reasons),
                        "power_w_max": max(pw) if pw else None, "samples": len(sm)})
        return out


# ------------------------------------------------------------------------------------------------ our arm
def ours_arm(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io, distributed as qdist
    from workloads import make_workload

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    pkg.load_library()  # fails loudly if the CUDA library is missing: there is no fallback

    # weak scaling: every rank owns its own batch of molecules (same shapes, rank-dependent seed not needed:
    # throughput does not depend on the values); the normal equations are summed over ranks each step.
    w = make_workload(args.config, n_mol=args.n_mol, D=args.D)
    dp = workload_io.device_problem(w, dev)
    p, D, n_mol, n_atoms = dp.params, w.model.D, w.n_mol, w.n_atoms
    rows = n_mol + 3 * n_atoms
    A = torch.empty((rows, D), dtype=torch.float32, device=dev)
    Z, G = A[:n_mol], A[n_mol:]
    ZtZ = torch.empty((D, D), dtype=torch.float32, device=dev)
    Zty = torch.empty((D,), dtype=torch.float32, device=dev)
    E = torch.empty((n_mol,), dtype=torch.float32, device=dev)
    F = torch.empty((n_atoms, 3), dtype=torch.float32, device=dev)

    def step(d):
        pkg.qmll_sorf_forward(p, d.x, d.elem, d.mol_off, d.grad, Z=Z, G=G)
        pkg.qmll_normal_equations(A, d.y, ZtZ=ZtZ, Zty=Zty)
        qdist.allreduce_normal_equations(ZtZ, Zty)
        pkg.qmll_predict(p, d.x, d.elem, d.mol_off, d.alpha, d.grad, energies=E, forces=F)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step(dp)
    barrier()

    # ---- device-resident timing (value) --------------------------------------------------------------
    pkg.reset_launch_count()
    pkg.collect_normal_equations_kernel_ms()
    pkg.time_normal_equations_kernel(True)
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    parts = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    barrier()
    e0.record()
    for k in range(args.steps):
        parts[k][0].record()
        pkg.qmll_sorf_forward(p, dp.x, dp.elem, dp.mol_off, dp.grad, Z=Z, G=G)
        parts[k][1].record()
        pkg.qmll_normal_equations(A, dp.y, ZtZ=ZtZ, Zty=Zty)
        qdist.allreduce_normal_equations(ZtZ, Zty)
        parts[k][2].record()
        pkg.qmll_predict(p, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad, energies=E, forces=F)
        parts[k][3].record()
    e1.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = pkg.launch_count()
    ms_total = qdist.max_over_ranks(e0.elapsed_time(e1), dev)
    ms_step = ms_total / args.steps
    syrk_ms, syrk_n = pkg.collect_normal_equations_kernel_ms()
    pkg.time_normal_equations_kernel(False)
    fwd_ms = sum(pp[0].elapsed_time(pp[1]) for pp in parts) / args.steps
    ne_ms = sum(pp[1].elapsed_time(pp[2]) for pp in parts) / args.steps
    pred_ms = sum(pp[2].elapsed_time(pp[3]) for pp in parts) / args.steps

    # ---- end to end through the public API with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        # Steps are pipelined the way a training loop would be: while step k computes, the copy stream uploads the
        # inputs of step k+1 into the other device buffer set and a third stream downloads the results of step k-1.
        # Every step still uploads ALL its inputs from pinned host memory and downloads ALL its results.
        host = {k: torch.from_numpy(v).pin_memory() for k, v in workload_io.host_arrays(w).items()}
        dbuf = [{k: torch.empty_like(v, device=dev) for k, v in host.items()} for _ in range(2)]
        outs = [{"ZtZ": torch.empty((D, D), dtype=torch.float32, device=dev),
                 "Zty": torch.empty((D,), dtype=torch.float32, device=dev),
                 "E": torch.empty((n_mol,), dtype=torch.float32, device=dev),
                 "F": torch.empty((n_atoms, 3), dtype=torch.float32, device=dev)} for _ in range(2)]
        out_host = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in outs[0].items()}
        h2d = sum(v.numel() * v.element_size() for v in host.values())
        d2h = sum(v.numel() * v.element_size() for v in out_host.values())
        s_in, s_out, s_main = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.current_stream()
        ev_in = [torch.cuda.Event() for _ in range(2)]       # inputs of buffer b uploaded
        ev_done = [torch.cuda.Event() for _ in range(2)]     # compute on buffer b finished
        ev_out = [torch.cuda.Event() for _ in range(2)]      # results of buffer b downloaded

        def e2e_run(n_steps):
            for k in range(n_steps):
                b = k & 1
                with torch.cuda.stream(s_in):
                    if k >= 2:
                        s_in.wait_event(ev_done[b])           # step k-2 no longer reads this input set
                    for name, v in host.items():
                        dbuf[b][name].copy_(v, non_blocking=True)
                    ev_in[b].record(s_in)
                s_main.wait_event(ev_in[b])
                if k >= 2:
                    s_main.wait_event(ev_out[b])              # results of step k-2 have left this output set
                db, o = dbuf[b], outs[b]
                g = workload_io.device_grad(db, dev)
                pkg.qmll_sorf_forward(p, db["x"], db["elem"], db["mol_off"], g, Z=Z, G=G)
                pkg.qmll_normal_equations(A, db["y"], ZtZ=o["ZtZ"], Zty=o["Zty"])
                qdist.allreduce_normal_equations(o["ZtZ"], o["Zty"])
                pkg.qmll_predict(p, db["x"], db["elem"], db["mol_off"], dp.alpha, g, energies=o["E"], forces=o["F"])
                ev_done[b].record(s_main)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_done[b])
                    for name, v in o.items():
                        out_host[name].copy_(v, non_blocking=True)
                    ev_out[b].record(s_out)
            s_main.wait_stream(s_out)

        e2e_run(2)
        barrier()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        s_in.wait_event(t0)
        e2e_run(args.steps)
        t1.record()
        barrier()
        e2e_ms = qdist.max_over_ranks(t0.elapsed_time(t1), dev) / args.steps
        e2e = {"value": world * n_mol / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "note": "public API on pinned HOST buffers; uploads/downloads of neighbouring steps overlap compute"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (tcgen05 3xTF32 A^T A) ---------------------------------------
    pk = peaks()
    alg_flops = float(rows) * D * (D + 1)            # symmetric half, fp32-equivalent
    kern_ms = syrk_ms / max(syrk_n, 1)
    achieved = alg_flops / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0
    tf32_peak = 0.5 * pk["bf16_sustained"]           # nominal tf32 : bf16 = 1 : 2 (profiling guide)
    peak3 = tf32_peak / 3.0                          # three TF32 MMAs per fp32-equivalent product
    roofline = {"kernel": "syrk_tcgen05_kernel", "bound": "tensor", "achieved": achieved, "peak": peak3,
                "unit": "TFLOP/s", "frac": achieved / peak3, "traffic": None,
                "note": (f"achieved = rows*D*(D+1) fp32-equivalent flops per launch / CUDA-event time of the kernel "
                         f"({kern_ms:.3f} ms avg over {syrk_n} launches); peak = bf16 sustained "
                         f"({pk['source']}) x 0.5 (tf32) / 3 (3xTF32); share of step = {kern_ms / ms_step:.3f}"),
                "full_gemm_equiv_tflops": 2.0 * rows * D * D / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0}

    # traffic of that kernel from the committed ncu --set full capture (profiles/), per launch
    try:
        with open(os.path.join(ROOT, "profiles", "r1_traffic.json")) as f:
            roofline["traffic"] = json.load(f)["syrk_tcgen05_kernel"]["dram_bytes_per_launch"]
    except Exception:
        roofline["traffic"] = None
    roofline["algorithmic_bytes"] = 2.0 * 4 * rows * D + 4.0 * D * (D + 1) / 2   # hi+lo operands once + half of C
    # the SORF kernels are bound by plain fp32 ALU issue: lane-ops / s against 148 SM x 128 x clock
    L = (w.model.d).bit_length() - 1
    T = w.model.T
    alu_peak = 148 * 128 * 1.965e9
    cols = 3.0 * sum(int(c) ** 2 for c in (w.mol_off[1:] - w.mol_off[:-1]))
    fr_ops = cols * D * (T * L + 2) + n_atoms * D * (T * L + 3)
    pr_ops = n_atoms * D * (2 * T * L + 6)
    sorf_rooflines = {
        "forward_plus_force_rows": {"bound": "alu", "achieved": fr_ops / (fwd_ms * 1e-3) / 1e12, "peak": alu_peak / 1e12,
                                    "unit": "T lane-ops/s", "frac": fr_ops / (fwd_ms * 1e-3) / alu_peak,
                                    "note": "algorithmic fp32 lane-ops D*(T*log2 d + 2) per gradient column + forward; "
                                            "time = whole qmll_sorf_forward call (CUDA events)"},
        "predict": {"bound": "alu", "achieved": pr_ops / (pred_ms * 1e-3) / 1e12, "peak": alu_peak / 1e12,
                    "unit": "T lane-ops/s", "frac": pr_ops / (pred_ms * 1e-3) / alu_peak,
                    "note": "D*(2*T*log2 d + 6) lane-ops per atom; whole qmll_predict call incl. the HBM-bound contraction"}}

    line = {"metric": METRIC, "value": world * n_mol / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 (SORF), 3xTF32 with fp32 accumulate (ZtZ)",
            "data": "synthetic",
            "config": {"workload": f"{w.name}: {n_mol} x 21-atom C9H8O4 configurations per GPU, d={w.model.d}, "
                                   f"D={D}, T={w.model.T}, sigma={w.model.sigma}, dense gradient (21,128,21,3); "
                                   f"train rows {rows} + predict E+F",
                       "l2": "inputs larger than L2 (gradient 677 MB, A 2.1 GB); no explicit flush",
                       "parallelism": f"dp{world} (molecules sharded, one all-reduce of ZtZ/Zty per step)"},
            "breakdown_ms": {"forward_and_force_rows": fwd_ms, "normal_equations": ne_ms, "predict": pred_ms,
                             "syrk_kernel": kern_ms},
            "ztz_tflops_fp32_equiv_half": achieved, "us_per_atom_predict": pred_ms * 1e3 / n_atoms,
            "roofline": roofline, "sorf_rooflines": sorf_rooflines, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}

    if not args.no_cpu_baseline and world == 1:
        sample_mol = min(8, n_mol)
        dt, cores, ws = time_oracle(args.config, D, sample_mol, 1, 0)
        line["cpu_baseline"] = {"value": sample_mol / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{sample_mol} of {n_mol} molecules at full D={D}: forward + force rows + "
                                          f"FP64 A^T A on its {ws.n_mol + 3 * ws.n_atoms} rows + predict, "
                                          f"{dt:.1f} s of CPU work"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def report_configs(args):
    """Absolute numbers and roofline fractions for all five configs (north_star), device-resident inputs."""
    import torch
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io
    from workloads import make_workload
    pk = peaks()
    alu_peak = 148 * 128 * 1.965e9

    def tm(f, n):
        for _ in range(2):
            f()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            f()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    for name, part in (("c1", "train"), ("c2", "train"), ("c3", "train"), ("c4", "train"), ("c4", "infer"), ("c5", "train")):
        w = make_workload(name, part=part)
        dp = workload_io.device_problem(w)
        p, m = dp.params, w.model
        L, T, D, na, nm = m.d.bit_length() - 1, m.T, m.D, w.n_atoms, w.n_mol
        out = {"config": w.name, "n_mol": nm, "n_atoms": na, "d": m.d, "D": D}
        train = w.grad is not None and w.grad.layout == "dense" and part == "train"
        if name == "c3" or train:
            rows = nm + (3 * na if train else 0)
            A = torch.empty((rows, D), dtype=torch.float32, device="cuda")
            if train:
                t = tm(lambda: pkg.qmll_sorf_forward(p, dp.x, dp.elem, dp.mol_off, dp.grad, Z=A[:nm], G=A[nm:]), args.steps)
                cols = 3.0 * sum(int(c) ** 2 for c in (w.mol_off[1:] - w.mol_off[:-1]))
                ops = cols * D * (T * L + 2) + na * D * (T * L + 3)
            else:
                t = tm(lambda: pkg.qmll_sorf_forward(p, dp.x, dp.elem, dp.mol_off, Z=A), args.steps)
                ops = na * D * (T * L + 3)
            out["forward_ms"] = t
            out["forward_alu_frac"] = ops / (t * 1e-3) / alu_peak
            out["forward_molecules_per_s"] = nm / (t * 1e-3)
            ZtZ = torch.empty((D, D), dtype=torch.float32, device="cuda")
            Zty = torch.empty((D,), dtype=torch.float32, device="cuda")
            y = dp.y if dp.y is not None and dp.y.numel() == rows else torch.zeros(rows, device="cuda")
            pkg.time_normal_equations_kernel(True)
            pkg.collect_normal_equations_kernel_ms()
            t = tm(lambda: pkg.qmll_normal_equations(A, y, ZtZ=ZtZ, Zty=Zty), max(1, args.steps // 2))
            kms, kn = pkg.collect_normal_equations_kernel_ms()
            pkg.time_normal_equations_kernel(False)
            out["normal_equations_ms"] = t
            out["ztz_kernel_ms"] = kms / max(kn, 1)
            tf = rows * D * (D + 1.0) / (kms / max(kn, 1) * 1e-3) / 1e12
            out["ztz_tflops_fp32eq_half"] = tf
            out["ztz_frac_of_3xtf32_sustained"] = tf / (0.5 * pk["bf16_sustained"] / 3.0)
            del A, ZtZ
        if name != "c3":
            E = torch.empty((nm,), dtype=torch.float32, device="cuda")
            F = torch.empty((na, 3), dtype=torch.float32, device="cuda")
            t = tm(lambda: pkg.qmll_predict(p, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad, energies=E, forces=F), args.steps)
            gbytes = (w.grad.dense.nbytes if w.grad.layout == "dense" else w.grad.nbr_val.nbytes)
            out.update({"predict_ms": t, "predict_molecules_per_s": nm / (t * 1e-3), "predict_us_per_atom": t * 1e3 / na,
                        "predict_alu_frac": na * D * (2 * T * L + 6) / (t * 1e-3) / alu_peak,
                        "predict_gradient_stream_GBps_if_alone": gbytes / (t * 1e-3) / 1e9})
        print(json.dumps(out), flush=True)
        del dp, w
        pkg.release_workspaces()
        torch.cuda.empty_cache()


if __name__ == "__main__":
    a = parse()
    if a.report_configs:
        report_configs(a)
    elif a.impl == "reference":
        reference_arm(a)
    else:
        ours_arm(a)

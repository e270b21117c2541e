"""bench.py -- one "step" = one pass of the whole SORF hot path over one batch of
synthetic input shaped like BASELINE.json:configs[3] (drug-like flexible molecule, the largest single-GPU config that
exercises every call):
    qmll_sorf_forward (+G) on the 500 training configurations  ->  qmll_normal_equations on [Z; G] (41 000 rows,
    D = 16384)  ->  qmll_predict (E + F) on the 2000 inference configurations
Prints ONE JSON line (contract in the task statement; extra keys: roofline, sorf_rooflines, configs, cpu_baseline,
e2e, clocks).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
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
WORKLOAD = ("c4: {nt} training + {ni} inference configurations of a 27-atom C12H12N2O molecule per GPU, d=256, D=16384, "
            "T=3, sigma=16, dense gradient (27,256,27,3); step = forward+force rows -> normal equations on {rows} rows "
            "-> predict E+F on the inference set; molecules per step = {nt} + {ni}")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n-train", type=int, default=None, help="shrink the workload (debug only; invalid as a bench)")
    ap.add_argument("--n-infer", type=int, default=None, help="shrink the workload (debug only; invalid as a bench)")
    ap.add_argument("--D", type=int, default=None, help="shrink the workload (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config block (C2, C3, C5)")
    ap.add_argument("--only-config", default=None, choices=["c2", "c3", "c5", "fchl19_cell", "solve"],
                    help="run only this entry of the per-config block and print it (used for the ncu captures in profiles/)")
    ap.add_argument("--force-rows", default="auto", choices=["auto", "fwht", "mma", "mma2"],
                    help="how the force rows are computed (qmll_sorf_forward_mode); the bench line uses auto")
    return ap.parse_args()


def peaks():
    """Roofline denominators: the driver's MEASURED_PEAKS.json (HBM copy, cuBLAS bf16) and this repo's own
    measurement of what that file lacks (profiles/peaks_r2.json: FADD issue rate, TF32 GEMM)."""
    out = {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback",
           "fadd_per_s": 148 * 128 * 1.965e9, "fadd_source": "nominal 148 SM x 128 lanes x 1.965 GHz",
           "tf32_burst": None, "tf32_sustained": None}
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        out.update({"hbm_gbs": p["hbm_gbs"], "bf16_burst": p["bf16_tflops"], "bf16_sustained": p["bf16_tflops_sustained"],
                    "source": "measured"})
    path = os.path.join(ROOT, "profiles", "peaks_r2.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        out.update({"fadd_per_s": p["alu"]["0"]["per_s"], "fadd_source": "measured (profiles/peaks_r2.json, FADD loop on all SMs)",
                    "tf32_burst": p["tensor"]["tf32_tflops_burst"], "tf32_sustained": p["tensor"]["tf32_tflops_sustained"],
                    "mufu_per_s": p["alu"]["9"]["per_s"]})
        if "14" in p["alu"]:
            out["dmma_fma_per_s"] = p["alu"]["14"]["per_s"]
    return out


# ------------------------------------------------------------------------------------------------ oracle arm
def oracle_stages(wt, wi):
    """Seconds the FP64 oracle, as it stands, needs for each stage of the step on the sample workloads."""
    import numpy as np
    import oracle
    t0 = time.perf_counter()
    Z = oracle.forward_w(wt)
    G = oracle.force_rows_w(wt)
    t1 = time.perf_counter()
    A = np.concatenate([Z, G]).astype(np.float32)
    oracle.normal_equations(A, wt.y)
    t2 = time.perf_counter()
    oracle.predict_w(wi)
    t3 = time.perf_counter()
    return {"forward_force_rows_s": t1 - t0, "normal_equations_s": t2 - t1, "predict_s": t3 - t2}


def oracle_sample(D, n_train=1, n_infer=2):
    import oracle
    from workloads import make_workload
    oracle.build()
    wt = make_workload("c4", n_mol=n_train, D=D)
    wi = make_workload("c4", n_mol=n_infer, D=D, part="infer")
    return wt, wi, oracle.num_threads()


def describe_sample(wt, wi, D):
    return (f"{wt.n_mol} of 500 training + {wi.n_mol} of 2000 inference configurations of c4 at full D={D}: forward + "
            f"force rows, FP64 A^T A on their {wt.n_mol + 3 * wt.n_atoms} rows, predict E+F")


def extrapolate(st, wt, wi, n_train=500, n_infer=2000):
    """Linear extrapolation of the sampled stage times to the full step (every stage is linear in its row count)."""
    return (st["forward_force_rows_s"] * n_train / wt.n_mol + st["normal_equations_s"] * n_train / wt.n_mol +
            st["predict_s"] * n_infer / wi.n_mol)


def reference_arm(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    D = args.D or 16384
    wt, wi, cores = oracle_sample(D, 2, 8)
    for _ in range(min(args.warmup, 1)):
        oracle_stages(wt, wi)
    tot, st = 0.0, None
    for _ in range(args.steps):
        st = oracle_stages(wt, wi)
        tot += sum(st.values())
    dt = tot / args.steps
    val = (wt.n_mol + wi.n_mol) / dt
    sample = describe_sample(wt, wi, D)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD.format(nt=500, ni=2000, rows=41000) + "; oracle arm: a bounded sample per step",
                       "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "stage_seconds_on_sample": st,
                             "extrapolated_full_step_s": extrapolate(st, wt, wi), "extrapolation": "linear in rows, labelled"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """SM clock, power and throttle reasons DURING the timed region: an in-process NVML thread (20 ms period, first
    sample immediately), or -- if pynvml is missing -- an `nvidia-smi -lms 20` child (which needs ~0.5 s to start and
    returned no sample at all on a fresh box for a 1 s timed region)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        import threading
        self.rows, self.p, self.t, self.halt = [], None, None, threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            ids = [v for v in vis.split(",") if v.strip()]
            phys = int(ids[index]) if ids and all(v.strip().isdigit() for v in ids) and index < len(ids) else index
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            mx = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
            bits = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40, "sw_power_cap": 0x4}

            def loop():
                while not self.halt.is_set():
                    try:
                        r = int(get_reasons(h))
                        self.rows.append((float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)), mx,
                                          pynvml.nvmlDeviceGetPowerUsage(h) / 1e3, [n for n, b in bits.items() if r & b]))
                    except Exception:
                        pass
                    self.halt.wait(0.02)

            self.t = threading.Thread(target=loop, daemon=True)
            self.t.start()
            self.how = "nvml thread"
        except Exception:
            self.how = "nvidia-smi -lms 20"
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            try:
                self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                           "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                          stderr=subprocess.DEVNULL)
            except Exception:
                self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.t is not None:
            self.halt.set()
            self.t.join(timeout=2)
        elif self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
            self.f.flush()
            self.f.seek(0)
            for r in [r.strip().split(",") for r in self.f.read().strip().splitlines() if r.strip()]:
                try:
                    names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
                    self.rows.append((float(r[0]), float(r[1]), float(r[2]),
                                      [n for n, v in zip(names, r[3:7]) if v.strip().lower().startswith("active")]))
                except Exception:
                    continue
            self.f.close()
            os.unlink(self.f.name)
        if self.rows:
            sm = sorted(r[0] for r in self.rows)
            out.update({"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.rows[-1][1],
                        "reasons": sorted({n for r in self.rows for n in r[3]}),
                        "power_w_max": max(r[2] for r in self.rows), "samples": len(sm), "how": self.how})
        return out


# ------------------------------------------------------------------------------------------------ roofline arithmetic
def sorf_ops(w, train):
    """Algorithmic fp32 lane-operations: forward D*(T*log2 d + 3) per atom, force rows
    D*(T*log2 d + 2) per gradient column, predict D*(2*T*log2 d + 6) per atom."""
    m = w.model
    L, T, D = m.d.bit_length() - 1, m.T, m.D
    fwd = w.n_atoms * D * (T * L + 3.0)
    cols = 3.0 * sum(int(c) ** 2 for c in (w.mol_off[1:] - w.mol_off[:-1])) if train else 0.0
    return fwd, cols * D * (T * L + 2.0), w.n_atoms * D * (2.0 * T * L + 6.0)


def ne_roofline(rows, D, kern_ms, ms_step, pk, traffic):
    alg_flops = float(rows) * D * (D + 1)            # symmetric half, fp32-equivalent
    achieved = alg_flops / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0
    peak = pk["bf16_sustained"] / 3.0                # three f16 MMAs (hi*hi, hi*lo, lo*hi) per fp32-equivalent product
    r = {"kernel": "syrk_tcgen05_kernel<f16 split>", "bound": "tensor", "achieved": achieved, "peak": peak,
         "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
         "algorithmic_bytes": 4.0 * rows * D + 2.0 * D * (D + 1),
         "frac_of_burst_peak": achieved / (pk["bf16_burst"] / 3.0),
         "note": (f"achieved = rows*D*(D+1) fp32-equivalent flops per call / CUDA-event time of the tcgen05 kernel per call "
                  f"({kern_ms:.3f} ms, summed over its row panels, events on the launch stream inside the library); peak = cuBLAS bf16 "
                  f"SUSTAINED ({pk['source']}: the kernel is timed inside a long step) / 3 -- f16 and bf16 MMAs run at "
                  f"the same rate; against the burst figure the fraction is frac_of_burst_peak; share of step = "
                  f"{kern_ms / ms_step:.3f}"),
         "full_gemm_equiv_tflops": 2.0 * rows * D * D / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0}
    if pk["tf32_sustained"]:
        r["vs_3xtf32_peak_measured"] = achieved / (pk["tf32_sustained"] / 3.0)   # what north_star's 3xTF32 scheme could reach
    if r["frac"] > 1.05:
        r["warning"] = "fraction above 1: the denominator is a cuBLAS measurement under the power cap, not the pipe peak"
    return r


def load_traffic():
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.json")) as f:
            t = json.load(f)
        return t["syrk_tcgen05_kernel"]["dram_bytes_per_launch"]
    except Exception:
        return None


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

    # weak scaling: every rank owns its own batch of configurations (same shapes; throughput does not depend on the
    # values); the normal equations are summed over ranks each step (packed lower triangle, NCCL).
    wt = make_workload("c4", n_mol=args.n_train, D=args.D)
    wi = make_workload("c4", n_mol=args.n_infer, D=args.D, part="infer")
    dt_, di_ = workload_io.device_problem(wt, dev), workload_io.device_problem(wi, dev)
    p, D = dt_.params, wt.model.D
    n_train, n_infer = wt.n_mol, wi.n_mol
    rows = n_train + 3 * wt.n_atoms
    A = torch.empty((rows, D), dtype=torch.float32, device=dev)
    Z, G = A[:n_train], A[n_train:]
    ZtZ = torch.empty((D, D), dtype=torch.float32, device=dev)
    Zty = torch.empty((D,), dtype=torch.float32, device=dev)
    E = torch.empty((n_infer,), dtype=torch.float32, device=dev)
    F = torch.empty((wi.n_atoms, 3), dtype=torch.float32, device=dev)
    reducer = qdist.NormalEquationsReducer(D, dev) if world > 1 else None

    rows_mode = {"auto": pkg.ROWS_AUTO, "fwht": pkg.ROWS_FWHT, "mma": pkg.ROWS_MMA, "mma2": pkg.ROWS_MMA2}[args.force_rows]

    def step(tr, inf, ZtZ_, Zty_, E_, F_):
        pkg.qmll_sorf_forward(p, tr.x, tr.elem, tr.mol_off, tr.grad, Z=Z, G=G, force_rows_mode=rows_mode)
        pkg.qmll_normal_equations(A, tr.y, ZtZ=ZtZ_, Zty=Zty_)
        if reducer is not None:
            reducer.allreduce(ZtZ_, Zty_)
        pkg.qmll_predict(p, inf.x, inf.elem, inf.mol_off, inf.alpha, inf.grad, energies=E_, forces=F_)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step(dt_, di_, ZtZ, Zty, E, F)
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
        pkg.qmll_sorf_forward(p, dt_.x, dt_.elem, dt_.mol_off, dt_.grad, Z=Z, G=G, force_rows_mode=rows_mode)
        parts[k][1].record()
        pkg.qmll_normal_equations(A, dt_.y, ZtZ=ZtZ, Zty=Zty)
        if reducer is not None:
            reducer.allreduce(ZtZ, Zty)
        parts[k][2].record()
        pkg.qmll_predict(p, di_.x, di_.elem, di_.mol_off, di_.alpha, di_.grad, energies=E, forces=F)
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
        host_t = {k: torch.from_numpy(v).pin_memory() for k, v in workload_io.host_arrays(wt).items()}
        host_i = {k: torch.from_numpy(v).pin_memory() for k, v in workload_io.host_arrays(wi).items()}
        dbuf_t = [{k: torch.empty_like(v, device=dev) for k, v in host_t.items()} for _ in range(2)]
        dbuf_i = [{k: torch.empty_like(v, device=dev) for k, v in host_i.items()} for _ in range(2)]
        outs = [{"ZtZ": torch.empty((D, D), dtype=torch.float32, device=dev),
                 "Zty": torch.empty((D,), dtype=torch.float32, device=dev),
                 "E": torch.empty((n_infer,), dtype=torch.float32, device=dev),
                 "F": torch.empty((wi.n_atoms, 3), dtype=torch.float32, device=dev)} for _ in range(2)]
        out_host = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in outs[0].items()}
        h2d = sum(v.numel() * v.element_size() for v in list(host_t.values()) + list(host_i.values()))
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
                    for name, v in host_t.items():
                        dbuf_t[b][name].copy_(v, non_blocking=True)
                    for name, v in host_i.items():
                        dbuf_i[b][name].copy_(v, non_blocking=True)
                    ev_in[b].record(s_in)
                s_main.wait_event(ev_in[b])
                if k >= 2:
                    s_main.wait_event(ev_out[b])              # results of step k-2 have left this output set
                tb, ib, o = dbuf_t[b], dbuf_i[b], outs[b]
                gt_, gi_ = workload_io.device_grad(tb, dev), workload_io.device_grad(ib, dev)
                pkg.qmll_sorf_forward(p, tb["x"], tb["elem"], tb["mol_off"], gt_, Z=Z, G=G, force_rows_mode=rows_mode)
                pkg.qmll_normal_equations(A, tb["y"], ZtZ=o["ZtZ"], Zty=o["Zty"])
                if reducer is not None:
                    reducer.allreduce(o["ZtZ"], o["Zty"])
                pkg.qmll_predict(p, ib["x"], ib["elem"], ib["mol_off"], di_.alpha, gi_, energies=o["E"], forces=o["F"])
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
        e2e = {"value": world * (n_train + n_infer) / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "h2d_GBps": h2d / (e2e_ms * 1e-3) / 1e9,
               "note": "public API on pinned HOST buffers; uploads/downloads of neighbouring steps overlap compute; "
                       "the 5.6 GB of descriptor gradients per step make this PCIe-bound"}
        del dbuf_t, dbuf_i, outs, host_t, host_i
        torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines -----------------------------------------------------------------------------------------------
    pk = peaks()
    kern_ms = syrk_ms / args.steps          # per CALL: a call runs one tcgen05 launch per panel of <= 32768 rows
    roofline = ne_roofline(rows, D, kern_ms, ms_step, pk, load_traffic())
    fwd_ops, fr_ops, _ = sorf_ops(wt, True)
    _, _, pr_ops = sorf_ops(wi, False)
    sm_mhz = (clocks or {}).get("sm_mhz") or 0.0
    fadd = pk["fadd_per_s"]
    cols = 3.0 * sum(int(c) ** 2 for c in (wt.mol_off[1:] - wt.mol_off[:-1]))
    mma_flops = 2.0 * 2.0 * wt.model.d * D * cols        # W (d x d per stack) x columns, hi + lo passes, 2 flop per MAC
    sorf_rooflines = {
        "force_rows_tensor": {"bound": "tensor", "achieved": mma_flops / (fwd_ms * 1e-3) / 1e12, "peak": pk["bf16_sustained"],
                              "unit": "TFLOP/s", "frac": mma_flops / (fwd_ms * 1e-3) / 1e12 / pk["bf16_sustained"],
                              "note": "the force rows run on tcgen05 (explicit W of every (element, stack) x fp16 hi/lo columns): "
                                      "useful f16 flops 2*2*d*D per gradient column (column padding to 16 not counted) / the whole "
                                      "qmll_sorf_forward call (CUDA events, incl. forward, W build and column split); peak = cuBLAS "
                                      "bf16 sustained (" + pk["source"] + ")"},
        "forward_plus_force_rows": {"bound": "alu", "achieved": (fwd_ops + fr_ops) / (fwd_ms * 1e-3) / 1e12,
                                    "peak": fadd / 1e12, "unit": "T lane-ops/s", "frac": (fwd_ops + fr_ops) / (fwd_ms * 1e-3) / fadd,
                                    "note": "FWHT-EQUIVALENT rate: the fp32 lane-ops the register chain would need, D*(T*log2 d + 2) per "
                                            "gradient column + forward, / the same call time; peak = " + pk["fadd_source"] +
                                            ".  The tensor-core path is not bound by this roofline (it can exceed 1)"},
        "predict": {"bound": "alu", "achieved": pr_ops / (pred_ms * 1e-3) / 1e12, "peak": fadd / 1e12,
                    "unit": "T lane-ops/s", "frac": pr_ops / (pred_ms * 1e-3) / fadd,
                    "gradient_stream_GBps": wi.grad.dense.nbytes / (pred_ms * 1e-3) / 1e9,
                    "note": "D*(2*T*log2 d + 6) lane-ops per atom; whole qmll_predict call: the fused kernel also streams the "
                            "descriptor gradient once (gradient_stream_GBps, against hbm_gbs below)"},
        "hbm_gbs_peak": pk["hbm_gbs"], "sm_mhz_during_run": sm_mhz}

    n_mol_step = n_train + n_infer
    line = {"metric": METRIC, "value": world * n_mol_step / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": warm, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (SORF), f16 hi/lo split tensor MMA with fp32 accumulate (ZtZ, fp32-level accuracy)",
            "data": "synthetic",
            "config": {"workload": WORKLOAD.format(nt=n_train, ni=n_infer, rows=rows), "force_rows": args.force_rows,
                       "l2": "inputs larger than L2 (gradients 1.1 + 4.5 GB, A 2.7 GB); no explicit flush",
                       "parallelism": f"dp{world} (configurations sharded, one all-reduce of the packed lower triangle of ZtZ + Zty per step)"},
            "breakdown_ms": {"forward_and_force_rows": fwd_ms, "normal_equations": ne_ms, "predict": pred_ms,
                             "syrk_kernel": kern_ms},
            "ztz_tflops_fp32_equiv_half": roofline["achieved"], "us_per_atom_predict": pred_ms * 1e3 / wi.n_atoms,
            "roofline": roofline, "sorf_rooflines": sorf_rooflines, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks}

    if not args.no_configs and world == 1:
        # NEXT row f1 beside the line: alpha = (ZtZ + lambda I)^-1 Zty of the step's own normal equations (FP64 Cholesky)
        lam = 1e-6 * float(torch.diagonal(ZtZ).mean())
        pkg.qmll_solve(ZtZ, Zty, lam)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _, info = pkg.qmll_solve(ZtZ, Zty, lam)
        e1.record()
        torch.cuda.synchronize()
        sms = e0.elapsed_time(e1)
        line["solve"] = {"D": D, "lambda": lam, "ms": sms, "info": int(info.item()),
                         "fp64_tflops": (D ** 3 / 3.0) / (sms * 1e-3) / 1e12}
        if "dmma_fma_per_s" in pk:      # measured FP64 tensor-core (DMMA) rate: 2 flops per FMA
            line["solve"]["frac_of_fp64_peak"] = line["solve"]["fp64_tflops"] * 1e12 / (2.0 * pk["dmma_fma_per_s"])
            line["solve"]["fp64_peak_tflops"] = 2.0 * pk["dmma_fma_per_s"] / 1e12
    del A, ZtZ, dt_, di_
    pkg.release_workspaces()
    torch.cuda.empty_cache()
    if not args.no_configs and world == 1:
        line["configs"] = other_configs(pk, max(2, args.steps // 2), rows_mode)
    if not args.no_cpu_baseline and world == 1:
        st_wt, st_wi, cores = oracle_sample(D, 3, 16)
        st = oracle_stages(st_wt, st_wi)
        tot = sum(st.values())
        line["cpu_baseline"] = {"value": (st_wt.n_mol + st_wi.n_mol) / tot, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": describe_sample(st_wt, st_wi, D) + f", {tot:.1f} s of CPU work",
                                "stage_seconds_on_sample": st,
                                "extrapolated_full_step_s": extrapolate(st, st_wt, st_wi),
                                "extrapolation": "linear in rows (every stage is), labelled; not measured"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def other_configs(pk, reps, rows_mode=0, only=None):
    """Absolute numbers and the binding roofline fraction for the other timed configs (north_star): C2, C3, C5."""
    import torch
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io
    from workloads import make_workload
    fadd = pk["fadd_per_s"]

    def tm(f):
        for _ in range(2):
            f()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            f()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    out = {}
    for name in ("c2", "c3", "c5"):
        if only is not None and name != only:
            continue
        w = make_workload(name)
        dp = workload_io.device_problem(w)
        p, m = dp.params, w.model
        D, na, nm = m.D, w.n_atoms, w.n_mol
        train = name == "c2"
        fwd_ops, fr_ops, pr_ops = sorf_ops(w, train)
        o = {"n_mol": nm, "n_atoms": na, "d": m.d, "D": D}
        if name in ("c2", "c3"):
            rows = nm + (3 * na if train else 0)
            A = torch.empty((rows, D), dtype=torch.float32, device="cuda")
            if train:
                t = tm(lambda: pkg.qmll_sorf_forward(p, dp.x, dp.elem, dp.mol_off, dp.grad, Z=A[:nm], G=A[nm:],
                                                     force_rows_mode=rows_mode))
            else:
                t = tm(lambda: pkg.qmll_sorf_forward(p, dp.x, dp.elem, dp.mol_off, Z=A))
            o.update({"forward_ms": t, "forward_molecules_per_s": nm / (t * 1e-3)})
            if train and rows_mode != 1:    # force rows on the tensor cores: not an ALU fraction (it may exceed 1)
                o["forward_fwht_equivalent_ops_vs_fadd_peak"] = (fwd_ops + fr_ops) / (t * 1e-3) / fadd
                o["note"] = ("force rows run on tcgen05: the FWHT-equivalent lane-op rate is quoted against the FADD peak "
                             "only to compare with the register-FWHT route (a speed-up factor, not a roofline fraction)")
            else:
                o["forward_alu_frac"] = (fwd_ops + fr_ops) / (t * 1e-3) / fadd
            if not train:
                # row f4 variants: the same Z on the tensor cores (expanded W) and the dense-matrix RFF map of equal size
                Zm = torch.empty((nm, D), dtype=torch.float32, device="cuda")
                t = tm(lambda: pkg.qmll_sorf_forward_mma(p, dp.x, dp.elem, dp.mol_off, Z=Zm))
                cos_s = na * D / (t * 1e-3)
                Em = torch.empty((nm,), dtype=torch.float32, device="cuda")
                te = tm(lambda: pkg.qmll_energies(pkg.qmll_sorf_forward_mma(p, dp.x, dp.elem, dp.mol_off, Z=Zm), dp.alpha, energies=Em))
                o.update({"predict_energies_mma_ms": te, "predict_energies_mma_molecules_per_s": nm / (te * 1e-3)})
                o.update({"forward_mma_ms": t, "forward_mma_molecules_per_s": nm / (t * 1e-3),
                          "forward_mma_useful_f16_tflops": 2.0 * 2.0 * m.d * D * na / (t * 1e-3) / 1e12,
                          "forward_mma_cos_frac_of_mufu_peak": cos_s / pk.get("mufu_per_s", 4.3e12)})
                # the paper's own N_transform = 2 (L268, L278): the FWHT chain is a third shorter, the expanded-W map is not
                p2 = pkg.SorfParams(d=m.d, D=D, n_transform=2, n_elem=m.n_elem, sigma=m.sigma,
                                    signs=p.signs[:, :, :2, :].contiguous(), bias=p.bias)
                o["forward_T2_ms"] = tm(lambda: pkg.qmll_sorf_forward(p2, dp.x, dp.elem, dp.mol_off, Z=Zm))
                o["forward_mma_T2_ms"] = tm(lambda: pkg.qmll_sorf_forward_mma(p2, dp.x, dp.elem, dp.mol_off, Z=Zm))
                Wr = torch.randn((m.n_elem, D, m.d), dtype=torch.float32, device="cuda") / m.sigma
                t = tm(lambda: pkg.qmll_rff_forward(Wr, p.bias, dp.x, dp.elem, dp.mol_off, Z=Zm))
                o.update({"rff_forward_ms": t, "rff_useful_f16_tflops": 3.0 * 2.0 * m.d * D * na / (t * 1e-3) / 1e12})
                del Zm, Wr
            ZtZ = torch.empty((D, D), dtype=torch.float32, device="cuda")
            Zty = torch.empty((D,), dtype=torch.float32, device="cuda")
            pkg.time_normal_equations_kernel(True)
            pkg.collect_normal_equations_kernel_ms()
            t = tm(lambda: pkg.qmll_normal_equations(A, dp.y, ZtZ=ZtZ, Zty=Zty))
            kms, kn = pkg.collect_normal_equations_kernel_ms()
            pkg.time_normal_equations_kernel(False)
            kcall = kms / (2 + reps)             # tm() makes 2 warm-up + reps calls; a call = one launch per row panel
            tf = rows * D * (D + 1.0) / (kcall * 1e-3) / 1e12
            o.update({"normal_equations_ms": t, "ztz_kernel_ms": kcall, "ztz_launches_per_call": kn // (2 + reps),
                      "ztz_tflops_fp32eq_half": tf,
                      "ztz_tensor_frac": tf / (pk["bf16_sustained"] / 3.0)})
            del A, ZtZ
        if name != "c3":
            E = torch.empty((nm,), dtype=torch.float32, device="cuda")
            F = torch.empty((na, 3), dtype=torch.float32, device="cuda")
            t = tm(lambda: pkg.qmll_predict(p, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad, energies=E, forces=F))
            gbytes = w.grad.dense.nbytes if w.grad.layout == "dense" else w.grad.nbr_val.nbytes
            o.update({"predict_ms": t, "predict_molecules_per_s": nm / (t * 1e-3), "predict_us_per_atom": t * 1e3 / na,
                      "predict_alu_frac": pr_ops / (t * 1e-3) / fadd,
                      "predict_gradient_stream_frac_of_hbm": gbytes / (t * 1e-3) / 1e9 / pk["hbm_gbs"]})
        else:
            E = torch.empty((nm,), dtype=torch.float32, device="cuda")
            t = tm(lambda: pkg.qmll_predict(p, dp.x, dp.elem, dp.mol_off, dp.alpha, energies=E))
            o.update({"predict_energies_ms": t, "predict_molecules_per_s": nm / (t * 1e-3)})
        out[name] = o
        del dp, w
        pkg.release_workspaces()
        torch.cuda.empty_cache()
    if only is None or only == "fchl19_cell":
        out["fchl19_cell"] = fchl19_config(pk, tm)
    if only == "solve":
        out["solve"] = solve_config(pk, tm)
    return out


def fchl19_config(pk, tm):
    """NEXT row f3: coordinates -> FCHL19 (+ Jacobian) -> per-element projection -> energy + forces on a periodic
    water-like cell shaped like config 5 (Table V): 25^3 atoms, r_cut 4.8 A (44 neighbours on
    average, K = 64 slots), Table I parameters (rep = 720), d = 256, D = 32768."""
    import numpy as np
    import torch
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io
    from workloads import cell_geometry, make_model, projection_inputs
    g = cell_geometry(2, 25, r_list=4.8, K=64)
    fp = pkg.Fchl19Params(r_cut=4.8)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    r, e, idx, sh, mol_off = t(g.r), t(g.elem), t(g.nbr_idx), t(g.nbr_shift), t(g.mol_off)
    na, K = g.nbr_idx.shape
    d, D = 256, 32768
    model = make_model(20220605, d=d, D=D, T=3, sigma=8.0)
    params = workload_io.device_params(model, "cuda:0")
    U = t(projection_inputs(seed=78, counts=[1], rep=fp.rep, d=d).U)
    alpha = t((np.random.default_rng(5).standard_normal(D) / np.sqrt(D)).astype(np.float32))
    o = {"n_atoms": na, "K": K, "mean_neighbours": float((g.nbr_idx >= 0).sum(1).mean()), "rep": fp.rep, "d": d, "D": D}
    o["fchl19_rho_ms"] = tm(lambda: pkg.qmll_fchl19(fp, r, e, idx, sh))
    rho, jidx, jval, info = pkg.qmll_fchl19(fp, r, e, idx, sh, jacobian=True)
    assert int(info.item()) == 0
    holder = {}

    def with_jac():
        holder["out"] = None
        holder["out"] = pkg.qmll_fchl19(fp, r, e, idx, sh, jacobian=True)
    del rho, jidx, jval
    ms = tm(with_jac)
    rho, jidx, jval, _ = holder.pop("out")
    jb = jval.numel() * 4
    o.update({"fchl19_rho_jacobian_ms": ms, "jacobian_bytes": jb,
              "jacobian_write_frac_of_hbm": jb / (ms * 1e-3) / 1e9 / pk["hbm_gbs"]})
    x = torch.empty((na, d), dtype=torch.float32, device="cuda")
    dx = torch.empty((na, K + 1, d, 3), dtype=torch.float32, device="cuda")
    o["project_x_ms"] = tm(lambda: pkg.qmll_project(rho, e, U))
    x, _ = pkg.qmll_project(rho, e, U)
    o["project_neighbor_ms"] = tm(lambda: pkg.qmll_project_neighbor(jval, e, U, idx=jidx, grad_out=dx))
    grad = pkg.Grad.make_neighbor(jidx, dx)
    E = torch.empty((1,), dtype=torch.float32, device="cuda")
    F = torch.empty((na, 3), dtype=torch.float32, device="cuda")
    o["predict_ms"] = tm(lambda: pkg.qmll_predict(params, x, e, mol_off, alpha, grad, energies=E, forces=F))
    tot = o["fchl19_rho_jacobian_ms"] + o["project_x_ms"] + o["project_neighbor_ms"] + o["predict_ms"]
    o.update({"coordinates_to_forces_jacobian_route_ms": tot, "jacobian_route_us_per_atom": tot * 1e3 / na})
    del jval, dx, grad
    torch.cuda.empty_cache()
    # the Jacobian-free backward pass (L268): rho -> x -> (E, dE/dx) -> dE/drho -> forces
    o["backward_g_ms"] = tm(lambda: pkg.qmll_sorf_backward_g(params, x, e, mol_off, alpha))
    _, gx = pkg.qmll_sorf_backward_g(params, x, e, mol_off, alpha)
    o["project_back_ms"] = tm(lambda: pkg.qmll_project_back(gx, e, U))
    wv = pkg.qmll_project_back(gx, e, U)
    o["fchl19_backward_ms"] = tm(lambda: pkg.qmll_fchl19_backward(fp, r, e, idx, wv, nbr_shift=sh, forces=F))
    tot = o["fchl19_rho_ms"] + o["project_x_ms"] + o["backward_g_ms"] + o["project_back_ms"] + o["fchl19_backward_ms"]
    o.update({"coordinates_to_forces_ms": tot, "us_per_atom": tot * 1e3 / na})
    pkg.release_workspaces()
    torch.cuda.empty_cache()
    return o


def solve_config(pk, tm, D=16384):
    """qmll_solve alone on a synthetic SPD system of the bench step's size (Gram matrix of a seeded Gaussian A with
    D + 512 rows; the bench line's own `solve` entry uses the step's ZtZ instead)."""
    import torch
    import paper_2206_01580_b200 as pkg
    g = torch.Generator(device="cuda").manual_seed(16384)
    A = torch.randn((D + 512, D), device="cuda", generator=g) / D ** 0.5
    ZtZ = A.T @ A
    Zty = torch.randn((D,), device="cuda", generator=g)
    del A
    lam = 1e-3
    ms = tm(lambda: pkg.qmll_solve(ZtZ, Zty, lam))
    alpha, info = pkg.qmll_solve(ZtZ, Zty, lam)
    res = ((ZtZ.double() @ alpha.double() + lam * alpha.double() - Zty.double()).norm() / Zty.double().norm()).item()
    o = {"D": D, "lambda": lam, "ms": ms, "info": int(info.item()), "relative_residual_fp32_alpha": res,
         "fp64_tflops": (D ** 3 / 3.0) / (ms * 1e-3) / 1e12}
    if "dmma_fma_per_s" in pk:
        o["frac_of_fp64_peak"] = o["fp64_tflops"] * 1e12 / (2.0 * pk["dmma_fma_per_s"])
    pkg.release_workspaces()
    torch.cuda.empty_cache()
    return o


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start N ranks of this script under torch.distributed.run."""
    argv = [a for a in sys.argv[1:]]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + argv
    sys.exit(subprocess.call(cmd))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        reference_arm(a)
    elif a.only_config:
        print(json.dumps({"configs": other_configs(peaks(), max(2, a.steps // 2), only=a.only_config)}))
    elif a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(a)
    else:
        ours_arm(a)

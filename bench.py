#!/usr/bin/env python
"""bench.py -- Helmholtz-apply throughput (GDoF/s, fp64) of libnk on B200, with the roofline fraction of
the kernel and the CPU oracle timed beside it.  Contract: see DESIGN.md section 8.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1|cfg2[:P]|cfg3[:P]|cfg4:P|cfg5[:P]] [--impl reference]

A step = one pass of the whole hot path (ONE fused kernel per block) over the
workload's mesh.  N > 1 (torchrun): every rank owns a mesh of the same size (elements are independent,
no collective in the data path) -> weak scaling.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from workloads import configs as cfgs          # noqa: E402  (data generators only)
from workloads import synthetic as wl          # noqa: E402

METRIC = "Helmholtz apply GDoF/s (fp64)"
HBM_FALLBACK_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
FP64_NOMINAL_TFLOPS = 37.2     # 148 SM x 64 DFMA/clk x 2 x 1.965 GHz


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--fields", type=int, default=1, help="multi-field block (P:199): N fields share one geometry; "
                    "single-block Helmholtz workloads only (DESIGN.md section 10)")
    ap.add_argument("--impl", default="nk", choices=["nk", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="budget of the cpu_baseline leg")
    return ap.parse_args()


def workload_blocks(name, device, rank=0):
    P = int(name.split(":")[1]) if ":" in name else None       # cfg4:P (and cfg2:P, cfg3:P, cfg5:P): the P-sweep
    title, op, blocks = cfgs.config_blocks(int(name[3:4]), device=device, P_sweep=P)
    for b in blocks:
        b["seed"] += 1000 * rank
    return title, op, blocks


def nmodes(shape, P):
    nm = P + 1
    return nm ** 3 if shape == 0 else nm * (nm + 1) * (nm + 2) // 6 if shape == 1 else nm * nm * (nm + 1) // 2


def algorithmic(shape, P, deformed, op="helmholtz"):
    """(bytes, flops) per element that the METHOD must move / compute."""
    nm, Q = P + 1, P + 2
    Nm, Nq = nmodes(shape, P), Q ** 3
    if shape == 0:
        bwd = 2 * (nm ** 3 * Q + nm ** 2 * Q ** 2 + nm * Q ** 3)
        chain = 0
    elif shape == 1:
        bwd = 2 * (Q * Nm + Q * Q * nm * (nm + 1) // 2 + nm * Q ** 3)
        chain = 9
    else:
        bwd = 2 * (Q * Nm + Q * Q * nm * nm + nm * Q ** 3)
        chain = 4
    if op == "mass":
        if shape == 0 and not deformed:      # affine hex: three nm x nm contractions in coefficient space
            return 16 * Nm + 8, 6 * nm ** 4 + Nm
        return 16 * Nm + 8 * (Nq if deformed else 1), 2 * bwd + Nq
    if shape == 0 and not deformed and P <= 7:
        # affine hex Laplacian / Helmholtz in coefficient space (P <= 7): 17 nm x nm contractions per line set
        return 16 * Nm + 56, 2 * 17 * nm ** 4 + 12 * Nm
    return 16 * Nm + 56 * (Nq if deformed else 1), 2 * bwd + 12 * Q ** 4 + (17 + 2 * chain) * Nq


# ---------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """SM clock + throttle reasons during the timed region (NVML, 5 ms period)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.max_mhz, self.stop_flag, self.ok = [], set(), None, False, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.005)

    def result(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


def physical_gpu_index(local):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


# ---------------------------------------------------------------------------------------------
def oracle_leg(workload, budget_s, want_steps=None, warmup=0):
    """Times oracle/ (as it stands) on the host cores on a bounded sample of the workload.
    Returns dict(value GDoF/s, cores, sample, ms_per_step)."""
    from oracle import nk_oracle as o        # the one place bench.py executes oracle/
    title, op, blocks = workload_blocks(workload, "cpu")
    chunk = 512
    per_block = []
    for b in blocks:
        el = o.Element(b["shape"], b["P"], b["P"] + 2)
        ne = b["v0"].shape[0]
        take = min(ne, chunk)
        A, J = (wl.sinusoidal_factors(b["v0"][:take], b["E"][:take], el.xi) if b["deformed"]
                else wl.affine_factors(b["v0"][:take], b["E"][:take]))
        x = wl.coefficients(b["seed"], take, el.Nm).numpy()
        per_block.append((el, A.numpy(), J.numpy(), x, b["lam"], take))

    def one_pass():
        dof = 0
        for el, A, J, x, lam, take in per_block:
            o.helmholtz(el, A, J, lam, x)
            dof += take * el.Nm
        return dof

    t0 = time.perf_counter()
    dof = one_pass()
    t_pass = time.perf_counter() - t0
    if want_steps is None:
        reps = max(1, min(200, int(budget_s / max(t_pass, 1e-6))))
    else:
        reps = want_steps
        for _ in range(warmup):
            one_pass()
    t0 = time.perf_counter()
    for _ in range(reps):
        one_pass()
    dt = (time.perf_counter() - t0) / reps
    return {"value": dof / dt / 1e9, "unit": "GDoF/s", "cores": 1, "kind": "oracle",
            "sample": "first %d elements of each block of %s, %d passes (numpy einsum, 1 thread)" % (chunk, title, reps),
            "ms_per_step": dt * 1e3, "title": title}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = max(1, min(args.steps, 50))
    r = oracle_leg(args.workload, args.cpu_seconds, want_steps=steps, warmup=min(args.warmup, 3))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": "GDoF/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 3), "ms_per_step": r["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": r["title"], "note": "plain CPU oracle (oracle/nk_oracle.py) on a bounded sample"},
            "cpu_baseline": {"value": r["value"], "unit": "GDoF/s", "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": "GDoF/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libnk has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    import paper_2606_20917_b200 as nk       # fails loudly if libnk.so is missing

    title, op, blocks = workload_blocks(args.workload, dev, rank)
    NSETS = 4   # rotate coefficient buffers so that an "HBM" number is not an L2 number
    work, dof, alg_bytes, alg_flops, geom_bytes = [], 0, 0, 0, 0
    for b in blocks:
        basis = nk.Basis(b["shape"], b["P"])
        A, J = cfgs.block_factors(b, basis.points())
        geom = nk.Geom(basis, A, J, b["deformed"], streams=nk.Geom.METRIC)
        ne = J.shape[0]
        del A, J
        xs = [wl.coefficients(b["seed"] + s, ne, basis.num_modes).to(dev) for s in range(NSETS)]
        ys = [torch.empty_like(xs[0]) for _ in range(NSETS)]
        work.append((basis, geom, xs, ys, b["lam"], ne))
        by, fl = algorithmic(b["shape"], b["P"], b["deformed"], "helmholtz")
        if op == "mass+laplacian":          # config 4: one mass and one Laplacian launch per step
            bm, fm = algorithmic(b["shape"], b["P"], b["deformed"], "mass")
            by, fl = by + bm, fl + fm
        nf = args.fields
        dof += ne * basis.num_modes * nf
        alg_bytes += (by + 16 * basis.num_modes * (nf - 1)) * ne      # the geometry is shared by the fields
        alg_flops += fl * ne * nf
        geom_bytes += 56 * ne * (basis.num_points if b["deformed"] else 1)
    torch.cuda.empty_cache()
    lam = blocks[0]["lam"]
    fxs = fys = None
    if args.fields > 1:
        if len(work) != 1 or op != "helmholtz":
            raise SystemExit("--fields applies to single-block Helmholtz workloads")
        basis, geom, xs, ys, _, ne = work[0]
        # two rotating sets of N fields each
        fxs = [[wl.coefficients(blocks[0]["seed"] + 10 * r + f, ne, basis.num_modes).to(dev) for f in range(args.fields)]
               for r in range(2)]
        fys = [[torch.empty_like(fxs[0][0]) for f in range(args.fields)] for r in range(2)]

    def step(i):
        s = i % NSETS
        if op == "mass+laplacian":
            for basis, geom, xs, ys, _, _ in work:
                nk.mass_apply(basis, geom, xs[s], ys[s])
                nk.laplacian_apply(basis, geom, xs[s], ys[(s + 1) % NSETS])
        elif len(work) == 1 and args.fields > 1:
            basis, geom, xs, ys, l, _ = work[0]
            nk.helmholtz_apply_fields(basis, geom, l, fxs[s % 2], fys[s % 2])
        elif len(work) == 1:
            basis, geom, xs, ys, l, _ = work[0]
            nk.helmholtz_apply(basis, geom, l, xs[s], ys[s])
        else:
            nk.helmholtz_apply_blocks([(w[0], w[1], w[2][s], w[3][s]) for w in work], lam)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(max(args.warmup, 3)):
        step(i)
    barrier()
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = nk.launch_count()
    barrier()
    torch.cuda.nvtx.range_push("nk_timed")     # lets `ncu --nvtx --nvtx-include "nk_timed/"` list exactly these launches
    e0.record()
    for i in range(args.steps):
        step(i)
    e1.record()
    torch.cuda.nvtx.range_pop()
    barrier()
    launches = nk.launch_count() - n0
    ms = e0.elapsed_time(e1)
    sampler.stop_flag = True
    sampler.join()
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = dof * world / (ms_step * 1e-3) / 1e9

    # ---- config 4: mass and Laplacian timed separately (locates the bandwidth / compute crossover) ----
    per_op = None
    if op == "mass+laplacian":
        per_op = {}
        basis, geom, xs, ys, _, ne = work[0]
        b0 = blocks[0]
        for name, fn in (("mass", nk.mass_apply), ("laplacian", nk.laplacian_apply)):
            for i in range(3):
                fn(basis, geom, xs[i % NSETS], ys[i % NSETS])
            barrier()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record()
            for i in range(args.steps):
                fn(basis, geom, xs[i % NSETS], ys[i % NSETS])
            t1.record()
            barrier()
            ms1 = t0.elapsed_time(t1) / args.steps
            bb, ff = algorithmic(b0["shape"], b0["P"], b0["deformed"], "mass" if name == "mass" else "helmholtz")
            if name == "laplacian" and b0["deformed"]:
                ff -= 2 * basis.num_points
            per_op[name] = {"ms": ms1, "gdofs": ne * basis.num_modes / (ms1 * 1e-3) / 1e9,
                            "alg_gbs": bb * ne / (ms1 * 1e-3) / 1e9, "alg_tflops": ff * ne / (ms1 * 1e-3) / 1e12}

    # ---- end to end: HOST buffers through nk_helmholtz_apply_host (H2D + kernel + D2H per step) ----
    e2e = None
    if op == "helmholtz" and args.fields == 1:
        hx = [[x.cpu().pin_memory() for x in w[2][:2]] for w in work]
        hy = [[torch.empty_like(h) for h in hs] for hs in hx]
        hy = [[h.pin_memory() for h in hs] for hs in hy]

        def e2e_step(i):
            for k, w in enumerate(work):
                nk.helmholtz_apply_host(w[0], w[1], w[4], hx[k][i % 2], hy[k][i % 2])

        esteps = max(3, min(args.steps, 30))
        for i in range(3):
            e2e_step(i)
        barrier()
        t0 = time.perf_counter()
        for i in range(esteps):
            e2e_step(i)
        barrier()
        dt = torch.tensor([(time.perf_counter() - t0) / esteps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        nbytes = sum(w[5] * w[0].num_modes * 8 for w in work)
        e2e = {"value": dof * world / float(dt.item()) / 1e9, "unit": "GDoF/s", "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": esteps,
               "note": "coefficients in pinned host memory -> nk_helmholtz_apply_host -> result in host memory; "
                       "geometry stream resident (uploaded once by nk_geom_upload)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel ----
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", HBM_FALLBACK_GBS))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback of B200_PROFILING.md"
    fp64_tf, _ = nk.probe_fp64_peak(400)
    ach_gbs = alg_bytes / (ms_step * 1e-3) / 1e9
    ach_tf = alg_flops / (ms_step * 1e-3) / 1e12
    hbm_frac, fp_frac = ach_gbs / hbm_peak, ach_tf / fp64_tf
    traffic = None
    tfile = os.path.join(ROOT, "profiles", "traffic_%s.csv" % args.workload.replace(":", "_P"))
    if os.path.exists(tfile):
        try:
            with open(tfile) as f:
                traffic = float(f.read().strip().splitlines()[-1].split(",")[-1])
        except Exception:
            traffic = None
    if hbm_frac >= fp_frac:
        roof = {"bound": "hbm", "achieved": ach_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_frac,
                "traffic": traffic, "peak_source": hbm_src}
    else:
        roof = {"bound": "alu", "achieved": ach_tf, "peak": fp64_tf, "unit": "TFLOP/s", "frac": fp_frac,
                "traffic": traffic, "peak_source": "nk_probe_fp64_peak (register-only DFMA chains, this run)"}
    if per_op:
        for v in per_op.values():
            v["hbm_frac"], v["fp64_frac"] = v.pop("alg_gbs") / hbm_peak, v.pop("alg_tflops") / fp64_tf
        roof["per_op"] = per_op
    roof["other"] = {"hbm_frac": hbm_frac, "fp64_frac": fp_frac, "fp64_probe_tflops": fp64_tf,
                     "fp64_nominal_tflops": FP64_NOMINAL_TFLOPS, "algorithmic_bytes_per_launch": alg_bytes,
                     "algorithmic_flops_per_launch": alg_flops, "kernel_ms": ms_step / max(1, launches // args.steps)}

    cpu = oracle_leg(args.workload, args.cpu_seconds)
    cpu_baseline = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}

    line = {"metric": METRIC, "value": value, "unit": "GDoF/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": title + (" x %d fields" % args.fields if args.fields > 1 else ""), "op": op, "dof_per_gpu": dof, "lambda": lam,
                       "l2": "inputs larger than L2: geometry stream %.0f MB per step + %d rotating coefficient "
                             "buffer sets" % (geom_bytes / 1e6, NSETS),
                       "parallelism": "elements sharded, no collective (dp%d)" % world},
            "clocks": sampler.result(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roof, "cpu_baseline": cpu_baseline}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

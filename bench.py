#!/usr/bin/env python
"""bench.py -- Helmholtz-apply throughput (GDoF/s, fp64) of libnk on B200, with the roofline fraction of
the kernel and the CPU oracle timed beside it.  Contract: see DESIGN.md section 8.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1|cfg2[:P[:Q]]|cfg3[:P[:Q]]|cfg4:P[:Q]|cfg5[:P[:Q]]]
                    [--per-workload default|none] [--impl reference]

A step = one pass of the whole hot path (ONE fused kernel per block) over the
workload's mesh.  N > 1 (torchrun): every rank owns a mesh of the same size (elements are independent,
no collective in the data path) -> weak scaling.  The headline line is config 2; `roofline.per_workload`
carries the other configurations, timed in the same run with the same event protocol.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Helmholtz apply GDoF/s (fp64)"
HBM_FALLBACK_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
FP64_NOMINAL_TFLOPS = 37.2     # 148 SM x 64 DFMA/clk x 2 x 1.965 GHz
PER_WORKLOAD_DEFAULT = ("cfg3", "cfg3:7", "cfg3:8", "cfg5", "cfg5:8", "cfg4:1", "cfg4:4", "cfg4:7", "cfg4:10",
                        "cfg2:7", "cfg2:10", "cfg2:4:7", "cfg5:5:8", "cfg1", "cg")
# cfg2:4:7 and cfg5:5:8 run on kernels specialised at run time by NVRTC (Q = P+3: outside the prebuilt Q = P+2 table)


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
    ap.add_argument("--per-workload", default=None, help="'default' (the list of DESIGN.md section 8), 'none', or a "
                    "comma-separated list of workloads; default: 'default' for the headline workload at N = 1, else 'none'")
    ap.add_argument("--form", type=int, default=0, help="nk_set_affine_simplex_form: 0 auto, 1 sum-factorised, 2 reference-matrix")
    return ap.parse_args()


def workload_blocks(name, device, rank=0):
    from workloads import configs as cfgs          # data generators only
    parts = name.split(":")
    P = int(parts[1]) if len(parts) > 1 else None       # cfg4:P (and cfg2:P, cfg3:P, cfg5:P): the P-sweep
    title, op, blocks = cfgs.config_blocks(int(name[3:4]), device=device, P_sweep=P)
    for b in blocks:
        b["seed"] += 1000 * rank
        b["Q"] = b["P"] + 2
    if len(parts) > 2:                                   # cfgN:P:Q -- the same mesh with Q points per direction (kernels
        for b in blocks:                                 # outside the Q = P+2 table are specialised at run time)
            b["Q"] = int(parts[2])
            title = title.replace("Q%d" % (b["P"] + 2), "Q%d" % b["Q"])
    return title, op, blocks


def nmodes(shape, P):
    nm = P + 1
    return nm ** 3 if shape == 0 else nm * (nm + 1) * (nm + 2) // 6 if shape == 1 else nm * nm * (nm + 1) // 2


def algorithmic(shape, P, deformed, op="helmholtz", form=0, Q=None):
    """Per element: bytes the METHOD must move, the flops of SURVEY 8(d)'s sum-factorised chain (`flops`: the
    contract's algorithmic count) and the flops of the form that actually runs (`flops_run`; DESIGN.md section 5:
    the coefficient-space forms of the affine operators need fewer)."""
    nm, Q = P + 1, (P + 2 if Q is None else Q)
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
        by, fl = 16 * Nm + 8 * (Nq if deformed else 1), 2 * bwd + Nq
    elif op == "laplacian":
        by, fl = 16 * Nm + 56 * (Nq if deformed else 1), 2 * bwd + 12 * Q ** 4 + (15 + 2 * chain) * Nq
    else:
        by, fl = 16 * Nm + 56 * (Nq if deformed else 1), 2 * bwd + 12 * Q ** 4 + (17 + 2 * chain) * Nq
    run = fl
    if not deformed and shape == 0:
        if op == "mass":                 # three nm x nm contractions in coefficient space
            run = 6 * nm ** 4 + Nm
        elif P <= 7:                     # 17 nm x nm contractions per line set (nk_stage_lapkron.inc)
            run = 2 * 17 * nm ** 4 + 12 * Nm
    if not deformed and form != 1 and (shape == 1 or (shape == 0 and P == 1) or (shape == 2 and P <= 3)):
        nc = 1 if op == "mass" else 6 if op == "laplacian" else 7    # reference-matrix GEMM (nk_dense.cuh): tets, trilinear hexes
        run = 2 * nc * Nm * Nm
    return {"bytes": by, "flops": fl, "flops_run": run}


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
def oracle_leg(workload, budget_s, want_steps=None, warmup=0, chunk=256):
    """Times oracle/ (as it stands: oracle.parallel hands unchanged element chunks to nk_oracle.helmholtz) over ALL
    host cores on a bounded sample of the workload: the first `chunk x cores` elements of every block.
    Returns dict(value GDoF/s, cores, cpu, sample, ms_per_step); best of >= 3 passes, table construction excluded
    (one untimed warm-up pass builds the tables in every worker)."""
    from oracle import nk_oracle as o        # the one place bench.py executes oracle/
    from oracle import parallel as op_
    from workloads import synthetic as wl
    title, _, blocks = workload_blocks(workload, "cpu")
    cores = os.cpu_count() or 1
    per_block = []
    for b in blocks:
        el = o.Element(b["shape"], b["P"], b["Q"])
        take = min(b["v0"].shape[0], chunk * cores)
        A, J = (wl.sinusoidal_factors(b["v0"][:take], b["E"][:take], el.xi) if b["deformed"]
                else wl.affine_factors(b["v0"][:take], b["E"][:take]))
        x = wl.coefficients(b["seed"], take, el.Nm).numpy()
        per_block.append((b["shape"], b["P"], b["Q"], A.numpy(), J.numpy(), x, b["lam"], take, el.Nm))
    with op_.OraclePool(cores) as pool:
        def one_pass():
            dof = 0
            for shape, P, Q, A, J, x, lam, take, Nm in per_block:
                pool.apply("helmholtz", shape, P, Q, A, J, lam, x, chunk=max(1, -(-take // cores)), want_result=False)
                dof += take * Nm
            return dof

        one_pass()                            # untimed: spawns the workers' tables
        t0 = time.perf_counter()
        dof = one_pass()
        t_pass = time.perf_counter() - t0
        if want_steps is None:
            reps = max(3, min(200, int(budget_s / max(t_pass, 1e-6))))
        else:
            reps = max(1, want_steps)
            for _ in range(warmup):
                one_pass()
        times = []
        for _ in range(reps):
            t0 = time.perf_counter()
            one_pass()
            times.append(time.perf_counter() - t0)
    best, mean = min(times), sum(times) / len(times)
    return {"value": dof / best / 1e9, "unit": "GDoF/s", "cores": cores, "cpu": op_.cpu_model(), "kind": "oracle",
            "sample": "first %d elements of each block of %s (%d per core), best of %d passes; numpy einsum, one "
                      "process per core, numpy threads pinned to 1, tables built before timing"
                      % (chunk * cores, title, chunk, reps),
            "ms_per_step": best * 1e3, "ms_per_step_mean": mean * 1e3, "title": title}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = max(3, min(args.steps, 50))
    r = oracle_leg(args.workload, args.cpu_seconds, want_steps=steps, warmup=min(args.warmup, 3))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": "GDoF/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 3), "ms_per_step": r["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": r["title"], "note": "plain CPU oracle (oracle/nk_oracle.py) on a bounded sample, all host cores"},
            "cpu_baseline": {"value": r["value"], "unit": "GDoF/s", "cores": r["cores"], "cpu": r["cpu"], "kind": "oracle",
                             "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": "GDoF/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
NSETS = 4   # rotate coefficient buffers so that an "HBM" number is not an L2 number


class Workload:
    """One configuration resident on the device: bases, geometry streams, rotating coefficient buffers."""

    def __init__(self, nk, name, dev, rank, fields=1, form=0):
        import torch
        from workloads import configs as cfgs
        from workloads import synthetic as wl
        self.nk, self.name, self.fields = nk, name, fields
        self.title, self.op, self.blocks = workload_blocks(name, dev, rank)
        self.work, self.dof, self.geom_bytes = [], 0, 0
        self.alg = {"bytes": 0, "flops": 0, "flops_run": 0}
        self.per_block = []
        for b in self.blocks:
            basis = nk.Basis(b["shape"], b["P"], b["Q"])
            A, J = cfgs.block_factors(b, basis.points())
            geom = nk.Geom(basis, A, J, b["deformed"], streams=nk.Geom.METRIC)
            ne = J.shape[0]
            del A, J
            xs = [wl.coefficients(b["seed"] + s, ne, basis.num_modes).to(dev) for s in range(NSETS)]
            ys = [torch.empty_like(xs[0]) for _ in range(NSETS)]
            self.work.append((basis, geom, xs, ys, b["lam"], ne))
            ops = ("mass", "laplacian") if self.op == "mass+laplacian" else ("helmholtz",)
            blk = {"bytes": 0, "flops": 0, "flops_run": 0}
            for o_ in ops:
                a = algorithmic(b["shape"], b["P"], b["deformed"], o_, form, b["Q"])
                blk["bytes"] += (a["bytes"] + 16 * basis.num_modes * (fields - 1)) * ne     # the geometry is shared by the fields
                blk["flops"] += a["flops"] * ne * fields
                blk["flops_run"] += a["flops_run"] * ne * fields
            for k in self.alg:
                self.alg[k] += blk[k]
            blk.update(shape=b["shape"], P=b["P"], deformed=b["deformed"], nelem=ne, dof=ne * basis.num_modes * fields)
            self.per_block.append(blk)
            self.dof += ne * basis.num_modes * fields
            self.geom_bytes += 56 * ne * (basis.num_points if b["deformed"] else 1)
        torch.cuda.empty_cache()
        self.lam = self.blocks[0]["lam"]
        self.fxs = self.fys = None
        if fields > 1:
            if len(self.work) != 1 or self.op != "helmholtz":
                raise SystemExit("--fields applies to single-block Helmholtz workloads")
            basis, geom, xs, ys, _, ne = self.work[0]
            self.fxs = [[wl.coefficients(self.blocks[0]["seed"] + 10 * r + f, ne, basis.num_modes).to(dev) for f in range(fields)]
                        for r in range(2)]
            self.fys = [[torch.empty_like(self.fxs[0][0]) for f in range(fields)] for r in range(2)]

    def step(self, i):
        nk, s = self.nk, i % NSETS
        if self.op == "mass+laplacian":
            for basis, geom, xs, ys, _, _ in self.work:
                nk.mass_apply(basis, geom, xs[s], ys[s])
                nk.laplacian_apply(basis, geom, xs[s], ys[(s + 1) % NSETS])
        elif len(self.work) == 1 and self.fields > 1:
            basis, geom, xs, ys, l, _ = self.work[0]
            nk.helmholtz_apply_fields(basis, geom, l, self.fxs[s % 2], self.fys[s % 2])
        elif len(self.work) == 1:
            basis, geom, xs, ys, l, _ = self.work[0]
            nk.helmholtz_apply(basis, geom, l, xs[s], ys[s])
        else:
            nk.helmholtz_apply_blocks([(w[0], w[1], w[2][s], w[3][s]) for w in self.work], self.lam)


def timed(fn, steps, warmup, barrier):
    """W untimed calls, then exactly `steps` calls between two CUDA events on torch's current stream (the stream
    the binding launches on), a barrier + synchronize on both sides.  Returns ms per call."""
    import torch
    for i in range(max(warmup, 3)):
        fn(i)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for i in range(steps):
        fn(i)
    e1.record()
    barrier()
    return e0.elapsed_time(e1) / steps


def fractions(alg, ms, hbm_peak, fp64_tf):
    """roofline figures of one timed unit: algorithmic bytes and flops / measured time against the
    measured peaks, plus the same with the flops of the form that runs."""
    t = ms * 1e-3
    hbm = alg["bytes"] / t / 1e9 / hbm_peak
    fp = alg["flops"] / t / 1e12 / fp64_tf
    fpr = alg["flops_run"] / t / 1e12 / fp64_tf
    bound = "hbm" if hbm >= max(fp, fpr) else "alu"
    return {"bound": bound, "frac": hbm if bound == "hbm" else fp, "hbm_frac": hbm, "fp64_frac": fp, "fp64_frac_running_form": fpr}


def measure_cg(nk, dev, barrier):
    """the assembled Helmholtz system of config 2's mesh (32^3 deformed hexes, P4, lambda = 1, C0
    connectivity of workloads.assembly) solved by Jacobi-preconditioned CG to 1e-8; time per iteration (gather + fused
    elemental kernel + scatter + 3 dot products + 3 vector updates) and the assembled apply on its own."""
    import torch
    from workloads import assembly as asm
    from workloads import synthetic as wl
    n, P, lam = 32, 4, 1.0
    basis = nk.Basis(0, P)
    v0, E = wl.hex_mesh(n, device=dev)
    A, J = wl.sinusoidal_factors(v0, E, basis.points().to(dev))
    geom = nk.Geom(basis, A, J, True, streams=nk.Geom.METRIC)
    del A, J
    l2g, ng = asm.hex_l2g(n, P)
    gs = nk.GatherScatter(l2g, ng)
    b = wl.coefficients(5, 1, ng).reshape(ng).to(dev)
    x = torch.zeros_like(b)
    nk.cg_solve(basis, geom, gs, lam, b, x, rtol=0.5, maxit=2)      # warm-up: builds the diagonal
    x.zero_()
    barrier()
    t0 = time.perf_counter()
    iters, rel = nk.cg_solve(basis, geom, gs, lam, b, x, rtol=1e-8, maxit=5000)
    barrier()
    dt = time.perf_counter() - t0
    y = torch.empty_like(b)
    ms_apply = timed(lambda i: nk.assembled_helmholtz_apply(basis, geom, gs, lam, b, y), 50, 3, barrier)
    out = {"workload": "CG on the assembled system of 32^3 deformed hexes P4 (%d global dofs, %d local)" % (ng, l2g.numel()),
           "iterations": iters, "relative_residual": rel, "ms_total": dt * 1e3, "ms_per_iteration": dt * 1e3 / max(iters, 1),
           "assembled_apply_ms": ms_apply, "assembled_apply_gdofs": ng / (ms_apply * 1e-3) / 1e9,
           "note": "wall clock around nk_cg_solve (it synchronises once per iteration to read the residual norm)"}
    del gs, geom
    torch.cuda.empty_cache()
    return out


def measure_cg_partitioned(nk, dev, rank, world, barrier):
    """The assembled Helmholtz system of config 2's mesh (32^3 deformed hexes, P4) split over the ranks by elements
    (workloads.assembly.partition_l2g) and solved by nk_part_cg_solve: every rank applies the fused kernel to its
    elements, the dofs on the cuts are summed by an NCCL all-reduce of the interface vector, dot products by scalar
    all-reduces (include/nk.h).  Strong scaling of ONE system; wall clock around the solve, max over ranks."""
    import torch
    import torch.distributed as dist
    from workloads import assembly as asm
    from workloads import synthetic as wl
    n, P, lam = 32, 4, 1.0
    basis = nk.Basis(0, P)
    l2g, ng = asm.hex_l2g(n, P)
    p = asm.partition_l2g(l2g, ng, world)[rank]
    del l2g
    lo, hi = p["range"]
    v0, E = wl.hex_mesh(n, device=dev)
    A, J = wl.sinusoidal_factors(v0[lo:hi].contiguous(), E[lo:hi].contiguous(), basis.points().to(dev))
    geom = nk.Geom(basis, A, J, True, streams=nk.Geom.METRIC)
    del A, J
    gs = nk.GatherScatter(p["l2g"], p["glob"].numel())
    part = nk.Partition(gs, p["shared_dof"], p["shared_slot"], p["shared_mult"], p["n_interface"], nk.torch_allreduce())
    b = wl.coefficients(wl.SEED0 + 77, 1, ng).reshape(ng)[p["glob"]].to(dev)         # consistent on the shared dofs
    x = torch.zeros_like(b)
    nk.part_cg_solve(basis, geom, part, lam, b, x, rtol=0.5, maxit=2, precond=nk.PRECOND_JACOBI)      # warm-up: diagonal, NCCL channels
    x.zero_()
    barrier()
    t0 = time.perf_counter()
    iters, rel = nk.part_cg_solve(basis, geom, part, lam, b, x, rtol=1e-8, maxit=20000, precond=nk.PRECOND_JACOBI)
    torch.cuda.synchronize()
    t = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return {"workload": "Jacobi-CG on the assembled system of 32^3 deformed hexes P4 (%d global dofs) split over %d rank(s)" % (ng, world),
            "ranks": world, "elements_per_rank": hi - lo, "interface_dofs": p["n_interface"], "iterations": iters,
            "relative_residual": rel, "ms_total": float(t.item()) * 1e3, "ms_per_iteration": float(t.item()) * 1e3 / max(iters, 1),
            "collectives_per_iteration": "1 interface all-reduce (%d doubles) + all-reduces of 1 and 2 doubles" % p["n_interface"],
            "note": "wall clock, max over ranks; the all-reduce is torch.distributed (NCCL) called back from nk_part_cg_solve"}


def measure_side_workload(nk, name, dev, rank, barrier, hbm_peak, fp64_tf, budget_ms=40.0, gpu_index=0):
    """One entry of roofline.per_workload: the workload timed with the protocol of the headline (CUDA events, >= 3
    warm-ups, rotating buffers), about `budget_ms` of kernel time -- the length of the headline's own timed region
    (400 x 0.08 ms = 33 ms): on this 1 kW part longer loops run into the power limiter (config 5: 20.8 GDoF/s over 40
    steps, 20.4 over 100, 19.3 over 400 with `sw_power_cap` and the SM clock at 1792 MHz), and the roofline
    denominators are burst figures.  Entries are separated by short pauses; SM clock and throttle reasons are sampled
    during each entry's timed region."""
    import torch
    if name == "cg":
        return measure_cg(nk, dev, barrier)
    time.sleep(0.2)     # let the power limiter recover from the previous entry
    w = Workload(nk, name, dev, rank)
    ms0 = timed(w.step, 3, 3, barrier)
    steps = int(max(20, min(2000, budget_ms / max(ms0, 1e-4))))
    sampler = ClockSampler(gpu_index)
    sampler.start()
    ms = timed(w.step, steps, 5, barrier)
    sampler.stop_flag = True
    sampler.join()
    out = {"workload": w.title, "op": w.op, "steps": steps, "ms": ms, "value": w.dof / (ms * 1e-3) / 1e9, "unit": "GDoF/s",
           "clocks": sampler.result(),
           "algorithmic_bytes": w.alg["bytes"], "algorithmic_flops": w.alg["flops"], "running_form_flops": w.alg["flops_run"]}
    out.update(fractions(w.alg, ms, hbm_peak, fp64_tf))
    if w.op == "mass+laplacian":          # config 4: each operator on its own, both flop counts (SURVEY 8(d) and the running form)
        basis, geom, xs, ys, _, ne = w.work[0]
        b0 = w.blocks[0]
        for opname, fn in (("mass", nk.mass_apply), ("laplacian", nk.laplacian_apply)):
            time.sleep(0.3)
            ms1 = timed(lambda i: fn(basis, geom, xs[i % NSETS], ys[i % NSETS]), steps, 3, barrier)
            a = algorithmic(b0["shape"], b0["P"], b0["deformed"], opname, 0, b0["Q"])
            a = {k: v * ne for k, v in a.items()}
            r = {"ms": ms1, "value": ne * basis.num_modes / (ms1 * 1e-3) / 1e9}
            r.update(fractions(a, ms1, hbm_peak, fp64_tf))
            out[opname] = r
    elif len(w.work) > 1:                  # config 5: each block's launch on its own
        out["blocks"] = []
        for (basis, geom, xs, ys, l, ne), blk in zip(w.work, w.per_block):
            time.sleep(0.3)
            smp = ClockSampler(gpu_index)
            smp.start()
            ms1 = timed(lambda i: nk.helmholtz_apply(basis, geom, l, xs[i % NSETS], ys[i % NSETS]), max(20, steps // 2), 3, barrier)
            smp.stop_flag = True
            smp.join()
            r = {"shape": ("hex", "tet", "prism")[blk["shape"]], "P": blk["P"], "nelem": ne, "ms": ms1,
                 "value": blk["dof"] / (ms1 * 1e-3) / 1e9, "clocks": smp.result()}
            r.update(fractions(blk, ms1, hbm_peak, fp64_tf))
            out["blocks"].append(r)
    if w.dof < 100000:                     # config 1 (64 elements): latency per call, eager and as a CUDA graph of 20 calls
        basis, geom, xs, ys, l, ne = w.work[0]
        out["us_per_call"] = ms * 1e3
        try:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                for i in range(3):
                    nk.helmholtz_apply(basis, geom, l, xs[i % NSETS], ys[i % NSETS])
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=side):
                    for i in range(20):
                        nk.helmholtz_apply(basis, geom, l, xs[i % NSETS], ys[i % NSETS])
            torch.cuda.current_stream().wait_stream(side)
            msg = timed(lambda i: graph.replay(), 100, 5, barrier)
            out["us_per_call_in_cuda_graph"] = msg * 1e3 / 20
        except Exception as ex:            # capture not available: report why, keep the eager figure
            out["us_per_call_in_cuda_graph"] = None
            out["cuda_graph_note"] = str(ex)[:200]
    del w
    torch.cuda.empty_cache()
    return out


def measure_e2e(nk, w, world, barrier, dev, steps):
    """End to end through nk_helmholtz_apply_host: pinned HOST coefficient buffers, H2D + kernel + D2H inside the timed
    region (wall clock around synchronising calls); geometry resident.  `cold` adds nk_geom_upload from host arrays."""
    import torch
    import torch.distributed as dist
    from workloads import configs as cfgs
    hx = [[x.cpu().pin_memory() for x in wk[2][:2]] for wk in w.work]
    hy = [[torch.empty_like(h).pin_memory() for h in hs] for hs in hx]

    def e2e_step(i):
        for k, wk in enumerate(w.work):
            nk.helmholtz_apply_host(wk[0], wk[1], wk[4], hx[k][i % 2], hy[k][i % 2])

    esteps = max(3, min(steps, 30))
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
    dt = float(dt.item())
    nbytes = sum(wk[5] * wk[0].num_modes * 8 for wk in w.work)
    e2e = {"value": w.dof * world / dt / 1e9, "unit": "GDoF/s", "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
           "steps": esteps, "ms_per_step": dt * 1e3, "pcie_gbs_per_direction": nbytes / dt / 1e9,
           "note": "coefficients in pinned host memory -> nk_helmholtz_apply_host -> result in host memory; "
                   "geometry stream resident (uploaded once by nk_geom_upload); copies and kernel overlap, so each "
                   "direction moves its bytes in the whole step time"}
    # cold: the geometry upload (host factors -> repack kernel -> metric stream) inside the timed region as well
    try:
        b0, wk0 = w.blocks[0], w.work[0]
        if len(w.work) == 1:
            A, J = cfgs.block_factors(b0, wk0[0].points())
            hA, hJ = A.cpu().pin_memory(), J.cpu().pin_memory()
            del A, J
            torch.cuda.empty_cache()
            times = []
            for i in range(3):
                barrier()
                t0 = time.perf_counter()
                g = nk.Geom(wk0[0], hA, hJ, b0["deformed"], streams=nk.Geom.METRIC)
                nk.helmholtz_apply_host(wk0[0], g, wk0[4], hx[0][i % 2], hy[0][i % 2])
                barrier()
                times.append(time.perf_counter() - t0)
                g.close()
            gbytes = hA.numel() * 8 + hJ.numel() * 8
            e2e["cold"] = {"value": w.dof / min(times) / 1e9, "unit": "GDoF/s", "ms": min(times) * 1e3,
                           "h2d_bytes": gbytes + nbytes, "d2h_bytes": nbytes,
                           "note": "one call of nk_geom_upload (host dxi/dx and detJ, pinned) + nk_helmholtz_apply_host, best of 3"}
    except Exception as ex:
        e2e["cold"] = {"value": None, "note": "not measured: %s" % str(ex)[:160]}
    return e2e


# ---------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libnk has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    under_torchrun = "RANK" in os.environ and "MASTER_ADDR" in os.environ
    if world > 1 or under_torchrun:
        dist.init_process_group("nccl", device_id=dev)
    import paper_2606_20917_b200 as nk       # fails loudly if libnk.so is missing
    if args.form:
        nk.set_affine_simplex_form(args.form)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = Workload(nk, args.workload, dev, rank, fields=args.fields, form=args.form)

    # ---- the timed region of the headline: W warm-ups, exactly K steps between two events, clocks sampled ----
    for i in range(max(args.warmup, 3)):
        w.step(i)
    barrier()
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = nk.launch_count()
    barrier()
    torch.cuda.nvtx.range_push("nk_timed")     # lets `ncu --nvtx --nvtx-include "nk_timed/"` list exactly these launches
    e0.record()
    for i in range(args.steps):
        w.step(i)
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
    ms_step = float(t.item()) / args.steps
    value = w.dof * world / (ms_step * 1e-3) / 1e9
    config = {"workload": w.title + (" x %d fields" % args.fields if args.fields > 1 else ""), "op": w.op,
              "dof_per_gpu": w.dof, "lambda": w.lam,
              "l2": "inputs larger than L2: geometry stream %.0f MB per step + %d rotating coefficient buffer sets"
                    % (w.geom_bytes / 1e6, NSETS),
              "parallelism": "elements sharded, no collective (dp%d)" % world}

    e2e = None
    if w.op == "helmholtz" and args.fields == 1:
        e2e = measure_e2e(nk, w, world, barrier, dev, args.steps)

    # the one path with a data-path collective: the assembled system on a mesh split over the ranks (NCCL all-reduce)
    cg_part = None
    if dist.is_initialized() and args.workload == "cfg2" and args.fields == 1:
        try:
            cg_part = measure_cg_partitioned(nk, dev, rank, world, barrier)
        except Exception as ex:
            cg_part = {"error": str(ex)[:300]}

    if rank != 0:
        if dist.is_initialized():
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
    dmma_tf, _ = nk.probe_fp64_dmma_peak(400)
    alg = dict(w.alg)
    fr = fractions(alg, ms_step, hbm_peak, fp64_tf)
    traffic, traffic_note = None, None
    tfile = os.path.join(ROOT, "profiles", "traffic_%s.csv" % args.workload.replace(":", "_P"))
    if os.path.exists(tfile):
        try:
            with open(tfile) as f:
                lines = f.read().strip().splitlines()
            traffic = float(lines[-1].split(",")[-1])
            traffic_note = "ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, from profiles/%s (%s)" % (
                os.path.basename(tfile), lines[0].lstrip("# "))
        except Exception:
            traffic = None
    if fr["bound"] == "hbm":
        roof = {"bound": "hbm", "achieved": alg["bytes"] / (ms_step * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": fr["hbm_frac"], "traffic": traffic, "peak_source": hbm_src}
    else:
        roof = {"bound": "alu", "achieved": alg["flops"] / (ms_step * 1e-3) / 1e12, "peak": fp64_tf, "unit": "TFLOP/s",
                "frac": fr["fp64_frac"], "traffic": traffic,
                "peak_source": "nk_probe_fp64_peak (register-only DFMA chains, this run); DMMA probe reads the same",
                "running_form": {"flops_per_launch": alg["flops_run"], "achieved": alg["flops_run"] / (ms_step * 1e-3) / 1e12,
                                 "frac": fr["fp64_frac_running_form"],
                                 "note": "flops of the coefficient-space form that runs (fewer than SURVEY 8(d)'s chain)"}}
    if traffic_note:
        roof["traffic_source"] = traffic_note
    roof["other"] = {"hbm_frac": fr["hbm_frac"], "fp64_frac": fr["fp64_frac"], "fp64_frac_running_form": fr["fp64_frac_running_form"],
                     "fp64_probe_tflops": fp64_tf, "fp64_dmma_probe_tflops": dmma_tf,
                     "fp64_nominal_tflops": FP64_NOMINAL_TFLOPS, "algorithmic_bytes_per_launch": alg["bytes"],
                     "algorithmic_flops_per_launch": alg["flops"], "running_form_flops_per_launch": alg["flops_run"],
                     "kernel_ms": ms_step / max(1, launches // args.steps)}

    # ---- the other configurations, same run, same protocol ----
    sel = args.per_workload
    if sel is None:
        sel = "default" if (world == 1 and args.workload == "cfg2" and args.fields == 1) else "none"
    names = PER_WORKLOAD_DEFAULT if sel == "default" else () if sel == "none" else tuple(s for s in sel.split(",") if s)
    if names:
        del w
        torch.cuda.empty_cache()
        pw = {}
        for name in names:
            try:
                pw[name] = measure_side_workload(nk, name, dev, rank, barrier, hbm_peak, fp64_tf, gpu_index=physical_gpu_index(local))
            except Exception as ex:
                pw[name] = {"error": str(ex)[:200]}
        roof["per_workload"] = pw
        try:
            k, cms = nk.jit_stats()
            roof["run_time_specialisation"] = {"kernels_compiled": int(k), "nvrtc_ms_total": cms,
                                               "note": "kernels outside the prebuilt Q = P+2 table (cfgN:P:Q entries), NVRTC on first use"}
        except Exception:
            pass
        roof["per_workload_note"] = ("each entry: W >= 3 warm-ups, `steps` launches between two CUDA events, 4 rotating "
                                     "buffer sets; frac = algorithmic bytes (hbm) or SURVEY 8(d) flops (alu) over the measured peak; "
                                     "fp64_frac_running_form counts the flops of the coefficient-space form that runs")

    cpu = oracle_leg(args.workload, args.cpu_seconds)
    cpu_baseline = {k: cpu[k] for k in ("value", "unit", "cores", "cpu", "kind", "sample")}

    line = {"metric": METRIC, "value": value, "unit": "GDoF/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config,
            "clocks": sampler.result(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roof, "cpu_baseline": cpu_baseline}
    if cg_part is not None:
        line["cg_partitioned"] = cg_part
    print(json.dumps(line), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py — headline measurement of the H / H^T pair.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config k]

One "step" = one pass of the whole hot path on one workload: data = H p0 followed by
image = H^T data (a single gradient evaluation) on BASELINE.json config 4 (512^3, 4000 samples,
4096 receivers) unless --config says otherwise.  Metric: Gcell-updates/s, where one call of H or
H^T performs nx*ny*nz*(nt-1) cell updates.  For N > 1 (torchrun) every rank runs an independent
replica of the workload on its own GPU ("replicas only"): value = all ranks' cell
updates / max-over-ranks device time.

Prints ONE JSON line on rank 0.  `--impl reference` times the fp64 CPU oracle instead (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gcell-updates/s for elastic FDTD forward+adjoint"
UNIT = "Gcell-updates/s"
B_ALG = 88.0          # algorithmic bytes per cell per time step (9 state R+W, 4 materials R)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1-based); 4 is the headline")
    ap.add_argument("--nt", type=int, default=None, help="development only: truncate the number of samples")
    ap.add_argument("--variant", type=int, default=0, help="kernel variant (0 = library default)")
    ap.add_argument("--acoustic", action="store_true",
                    help="SURVEY 8(f)-2: the config's medium with mu = 0 (H^dagger_{mu=0}, PAPER.md:299): fluid-only kernels, 44 B per cell-step")
    ap.add_argument("--pgd", action="store_true", help="SURVEY 8(f)-1: projected-gradient reconstruction (use with --config 5)")
    ap.add_argument("--iters", type=int, default=10, help="--pgd: iterations")
    ap.add_argument("--power-iters", type=int, default=8, help="--pgd: power iterations for the step size")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------
def workload_name(prob, args):
    p = prob.prm
    s = f"BASELINE config {args.config}: {p.nx}x{p.ny}x{p.nz}, nt={p.nt}, L={prob.L}, npml={p.npml}"
    if getattr(args, "acoustic", False):
        s += "; shear modulus set to zero (the paper's H_mu=0: fluid-only kernels)"
    if args.nt is not None:
        s += " (nt truncated: development run, not the headline)"
    return s


def make_problem(args):
    from paper_1709_02733_b200 import synth
    prob = synth.make_config(args.config, nt=args.nt)
    return synth.fluid_version(prob) if args.acoustic else prob


def bytes_per_cell_step(args):
    """Algorithmic bytes per cell per time step: elastic 9 state fields R+W + 4 materials R = 88;
    fluid-only 4 state fields R+W + 3 materials R = 44."""
    return 44.0 if args.acoustic else B_ALG


def cpu_sample(prob):
    """Bounded sample of the workload for the oracle: a block of the same volumes, few samples."""
    from paper_1709_02733_b200 import synth
    n_full = prob.prm.nx
    n = min(n_full, 160)
    nt = 200 if n_full > n else min(prob.prm.nt, 200)      # ~15-20 s of oracle work at 0.1 Gcell-updates/s
    if n_full > n:
        # block under the top of the hemispherical array: contains water, porous skull and receivers
        x0 = y0 = (n_full - n) // 2
        z0 = n_full - n - max(prob.prm.npml // 2, 1)
        sub = synth.crop(prob, (x0, y0, z0), n, nt)
        what = f"{n}^3 block at ({x0},{y0},{z0}) of the workload's volumes, nt={nt}, {sub.L} receivers, forward+adjoint"
    else:
        from dataclasses import replace
        sub = replace(prob, prm=replace(prob.prm, nt=nt))
        what = f"the full {n}^3 grid, nt={nt}, forward+adjoint"
    return sub, what


def time_oracle(sub, repeats=1):
    """Seconds for one forward + one adjoint of the oracle on `sub` (as it stands, OpenMP threads);
    best of `repeats`."""
    import numpy as np
    from oracle.oracle import Oracle, threads
    o = Oracle.from_problem(sub)
    p0 = sub.p0.astype(np.float64)
    best = float("inf")
    for _ in range(repeats):
        t = time.perf_counter()
        d = o.forward(p0)
        o.adjoint(d)
        best = min(best, time.perf_counter() - t)
    o.close()
    cells = 2.0 * sub.prm.N * (sub.prm.nt - 1)
    return best, cells, threads()


def run_reference(args):
    """`--impl reference`: the fp64 CPU oracle on a bounded sample of the arm's workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1709_02733_b200 import synth
    prob = make_problem(args)
    sub, what = cpu_sample(prob)
    for _ in range(max(args.warmup, 0) and 1):
        time_oracle(sub)
    t_tot, cells_tot = 0.0, 0.0
    cores = 1
    for _ in range(max(args.steps, 1)):
        t, cells, cores = time_oracle(sub)
        t_tot += t
        cells_tot += cells
    v = cells_tot / t_tot / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(prob, args), "sample": what},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if not self.proc:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        try:
            for ln in open(self.path):
                c = [v.strip() for v in ln.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); smax.append(float(c[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(smax), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def max_over_ranks(value, world, device=None):
    """MAX of a per-rank scalar over all ranks (the slowest rank defines the time of a multi-GPU step).
    Uses the default process group (NCCL on GPUs; gloo in the CPU tests); identity for world = 1."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(cells_per_rank_step, steps, world, ms_max):
    """Replicas only: every rank processes its own copy of the workload, so the job's cell updates are
    world x (one rank's), divided by the slowest rank's device time.  Gcell-updates/s."""
    return world * cells_per_rank_step * steps / (ms_max * 1e-3) / 1e9


def csrc_digest():
    """sha256 over the CUDA sources: a committed ncu capture is only quoted while the kernels it measured
    are the kernels that run."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1709_02733_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def committed_traffic(config):
    """DRAM bytes per launch from the committed `ncu --set full` capture (profiles/traffic.txt), or (None, why).
    Not measured in this run: the JSON line says so in `traffic_source`."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    if not os.path.exists(path):
        return None, "no committed capture (profiles/traffic.txt)"
    try:
        rec = json.load(open(path))
        t = rec.get(f"config{config}")
        if not t:
            return None, f"profiles/traffic.txt has no capture of config {config}"
        if rec.get("csrc_sha256_16") != csrc_digest():
            return None, "profiles/traffic.txt is stale: the kernel sources changed after the capture (%s)" % rec.get("captured")
        return t, "profiles/traffic.txt: ncu --set full capture of %s, kernel sources %s (not measured in this run)" % (
            rec.get("captured"), rec.get("csrc_sha256_16"))
    except Exception as e:      # a broken record is no record
        return None, f"profiles/traffic.txt unreadable: {e}"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def run_pgd(args):
    """SURVEY 8(f)-1 / BASELINE config 5: d = H p_true + 1 % seeded Gaussian noise, step 1/||H||^2 from a power
    iteration, then `--iters` iterations of p <- max(0, p - s H^T (H p - d)) through pact_pgd, one call per iteration
    so that each is timed (CUDA events on the library's stream) and its image error is read.  One JSON line."""
    import numpy as np
    import torch
    from paper_1709_02733_b200 import build, synth
    from paper_1709_02733_b200.binding import Pact
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    build.build()
    prob = make_problem(args)
    prm = prob.prm
    ctx = Pact.from_problem(prob, device=dev)
    ctx.set_option("variant", args.variant)
    ctx.set_option("check_finite", 1)
    rng = np.random.default_rng(170902733 + 100 * args.config)
    p_true = torch.from_numpy(np.ascontiguousarray(prob.p0, dtype=np.float32)).to(dev)
    d = ctx.forward(p_true)
    noise = torch.from_numpy(rng.standard_normal((prm.nt, prob.L)).astype(np.float32)).to(dev)
    d = d + 0.01 * float(d.abs().max()) * noise
    del noise
    v = torch.from_numpy(rng.standard_normal(ctx.shape).astype(np.float32)).to(dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    e0, e1 = ev(), ev()
    e0.record(ctx.stream)
    sigma2 = ctx.power_iteration(v, args.power_iters)
    e1.record(ctx.stream)
    torch.cuda.synchronize(dev)
    t_power = e0.elapsed_time(e1) * 1e-3
    step = 1.0 / sigma2
    p = torch.zeros(ctx.shape, dtype=torch.float32, device=dev)
    nt2 = float(p_true.double().norm())
    times, err, res, upd = [], [], [], []
    clocks = ClockSampler(dev.index or 0)
    clocks.start()
    for k in range(args.iters):
        a, b = ev(), ev()
        a.record(ctx.stream)
        r, u = ctx.pgd(p, d, step, 1)
        b.record(ctx.stream)
        torch.cuda.synchronize(dev)
        times.append(a.elapsed_time(b) * 1e-3)
        res.append(r[0]); upd.append(u[0])
        err.append(float((p.double() - p_true.double()).norm()) / nt2)
    clk = clocks.stop()
    cells_iter = 2.0 * prm.N * (prm.nt - 1)
    ts = sorted(times)
    med = ts[len(ts) // 2]
    line = {"metric": "seconds per projected-gradient iteration (one H and one H^T)", "value": med, "unit": "s",
            "n_gpus": 1, "steps": args.iters, "warmup": 0, "ms_per_step": 1e3 * med, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(prob, args) + "; d = H p_true + 1 % noise; p_0 = 0; step = 1/||H||^2",
                       "power_iterations": args.power_iters, "elided_material_planes": ctx.info("elided_material_planes")},
            "gcell_updates_per_s": cells_iter / med / 1e9, "sigma2": sigma2, "step": step, "power_iteration_s": t_power,
            "seconds_per_iteration": times, "relative_image_error": err, "residual_l2": res, "update_l2": upd,
            "data_l2": float(d.double().norm()), "clocks": clk,
            "gpu_launches": int(args.iters * (2 * (2 * (prm.nt - 1) + prm.nt) + 8))}
    print(json.dumps(line), flush=True)
    ctx.close()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.pgd:
        run_pgd(args)
        return
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1709_02733_b200 import build, synth
    from paper_1709_02733_b200.binding import Pact

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    build.build()

    prob = make_problem(args)                             # every rank: an independent replica
    prm = prob.prm
    ctx = Pact.from_problem(prob, device=dev)
    ctx.set_option("variant", args.variant)
    p0 = torch.from_numpy(prob.p0).to(dev)
    data = torch.empty((prm.nt, prob.L), dtype=torch.float32, device=dev)
    image = torch.empty(ctx.shape, dtype=torch.float32, device=dev)

    def step():
        ctx.forward(p0, out=data)        # data = H p0
        ctx.adjoint(data, out=image)     # image = H^T data

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        step()
    barrier()
    try:        # homogeneous (tile, plane) material boxes served from L2-resident palette planes (fused path only)
        elided = ctx.info("elided_material_planes")
    except Exception:
        elided = None
    ctx.set_option("profile", 1)         # CUDA events around sampled launches, on the library's stream
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    ev0.record(ctx.stream)
    for _ in range(args.steps):
        step()
    ev1.record(ctx.stream)
    torch.cuda.synchronize(dev)
    barrier()
    clk = clocks.stop() if rank == 0 else None
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
    cells_step = 2.0 * prm.N * (prm.nt - 1)                # forward + adjoint
    value = whole_job_rate(cells_step, args.steps, world, ms)

    # ---- look at what the timed steps produced: a blow-up must not print a throughput
    d64, i64 = data.double(), image.double()
    checks = {"finite": bool(torch.isfinite(data).all().item() and torch.isfinite(image).all().item()),
              "data_l2": float(d64.norm().item()), "image_l2": float(i64.norm().item()),
              "data_absmax": float(data.abs().max().item()), "image_absmax": float(image.abs().max().item())}
    del d64, i64
    assert checks["finite"], f"non-finite values in the result of the timed steps: {checks}"
    if args.nt is None:      # (a truncated development run may end before the wave reaches a receiver)
        assert checks["data_l2"] > 0.0 and checks["image_l2"] > 0.0, f"the timed steps produced zeros: {checks}"

    # ---- roofline of the step kernels, from the library's own CUDA events in the timed region
    loop_f, k_f, n_f = ctx.timing("forward")
    loop_a, k_a, n_a = ctx.timing("adjoint")
    ctx.set_option("profile", 0)
    launches = (sum(n_f.values()) + sum(n_a.values()) + 3) * args.steps   # + argument record x2 and tau per step
    # device time of one time step's kernels (all launches of the step, in the mix they ran)
    step_kinds_f = ("fwd_vel", "fwd_str", "fwd_fused", "fwd_slab", "fwd_interior")
    step_kinds_a = ("adj_a", "adj_b", "adj_fused", "adj_slab", "adj_interior")
    # sampled launches (CUDA events around every ~80th launch): a cross-check and the slab / interior split
    ts_fwd = sum(k_f[k] * n_f[k] for k in step_kinds_f) / max(prm.nt - 1, 1)
    ts_adj = sum(k_a[k] * n_a[k] for k in step_kinds_a) / max(prm.nt - 1, 1)
    # basis of the roofline: the whole time loop of the last timed forward / adjoint call (events on the library's
    # stream around the loop) divided by its nt - 1 steps.  It contains the receiver kernels (< 0.4 % of a step) and
    # no event overhead; the sampled per-launch times read a few per cent higher because every sampled launch
    # carries two event records and the launch gap.
    t_fwd = loop_f / max(prm.nt - 1, 1)
    t_adj = loop_a / max(prm.nt - 1, 1)
    peak, peak_src = peaks()
    pml_extra = (16.0 if args.acoustic else 48.0) * 3 * 2 * prm.npml / prm.nx if prm.npml else 0.0
    roof = None
    if t_fwd > 0 and t_adj > 0:
        B = bytes_per_cell_step(args)
        ach = 2 * B * prm.N / ((t_fwd + t_adj) * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                "peak_source": peak_src, "kernel": "step kernels of one forward + one adjoint time step",
                "basis": "time loop of the last timed forward / adjoint call / (nt - 1) steps, CUDA events on the library's stream",
                "sampled_forward_step_ms": ts_fwd, "sampled_adjoint_step_ms": ts_adj,
                "bytes_per_cell_step": B, "pml_bytes_per_cell_step_not_credited": pml_extra,
                "forward_step_ms": t_fwd, "adjoint_step_ms": t_adj,
                "forward_frac": B * prm.N / (t_fwd * 1e-3) / 1e9 / peak,
                "adjoint_frac": B * prm.N / (t_adj * 1e-3) / 1e9 / peak,
                "forward_loop_ms": loop_f, "adjoint_loop_ms": loop_a,
                "kernel_ms": {"forward": {k: v for k, v in k_f.items() if v}, "adjoint": {k: v for k, v in k_a.items() if v}}}
        t, src = committed_traffic(args.config)
        roof["traffic_source"] = src
        if t:
            # per launch of the dominant kernel (the adjoint step)
            pre = "acoustic_" if args.acoustic else ""
            roof["traffic"] = t[pre + "adjoint_bytes_per_launch"] / 1e9
            roof["traffic_unit"] = "GB per launch (dram__bytes_read.sum + dram__bytes_write.sum), algorithmic %.2f" % (B * prm.N / 1e9)
            roof["traffic_forward"] = t[pre + "forward_bytes_per_launch"] / 1e9

    # ---- end to end through the host-buffer entry points (pinned host memory, copies inside)
    e2e = None
    if not args.no_e2e:
        p0_h = torch.from_numpy(prob.p0).pin_memory()
        data_h = torch.empty((prm.nt, prob.L), dtype=torch.float32).pin_memory()
        image_h = torch.empty(ctx.shape, dtype=torch.float32).pin_memory()
        n_e2e = 1
        ctx.forward_host(p0_h, data_h); ctx.adjoint_host(data_h, image_h)     # warm (staging buffers)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            ctx.forward_host(p0_h, data_h)
            ctx.adjoint_host(data_h, image_h)
        torch.cuda.synchronize(dev)
        t_e = max_over_ranks(time.perf_counter() - t0, world, dev)
        nb = prm.N * 4 + prm.nt * prob.L * 4
        e2e = {"value": whole_job_rate(cells_step, n_e2e, world, t_e * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": nb, "d2h_bytes_per_step": nb, "steps": n_e2e,
               "api": "pact_forward_host + pact_adjoint_host (pinned host buffers)"}

    # ---- the oracle beside it (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sub, what = cpu_sample(prob)
        t, cells, cores = time_oracle(sub)
        cpu = {"value": cells / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what, "seconds": t}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(prob, args), "parallelism": "replicas only" if world > 1 else "single GPU",
                           "step": "one pact_forward + one pact_adjoint", "l2": "inputs larger than L2 (no flush needed)"
                           if ctx.device_bytes() > 4 * 126e6 else "working set near L2 size: latency/L2-bound case",
                           "variant": args.variant, "device_bytes": ctx.device_bytes(),
                           "elided_material_planes": elided},
                "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clk,
                "checks": checks}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

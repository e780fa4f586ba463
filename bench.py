"""bench.py - the headline measurement of the DGTD hot path (contract: DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2_two_layer]
                    [--timesteps T] [--no-extras]

One bench "step" = one whole pass of the hot path over one batch of synthetic input = T global time
steps (BASELINE.json config 2: T = 1000, single-rate AB3, fp32, N = 3, 98 304 tets) of
volume + surface right-hand side, point source and update, all enqueued by ONE C-ABI call dg_step(T).
value  = DOF-updates/s with the fields resident in HBM (CUDA events on the bound stream).
e2e    = the same through the C ABI with HOST buffers: dg_set_state(host q0) -> dg_step(T) ->
         dg_get_fields(host q), host<->device copies and layout conversion inside the timed region.
roofline = the dominant kernel of the step, timed live with one CUDA event pair per launch
         (dg_set_profiling) in a separate pass over the same steps.
cpu_baseline = the fp64 numpy oracle on the box's host cores on a bounded sample of the same workload.
--impl reference times that oracle (there is no reference implementation: the reference is a paper).
Multi-GPU (torchrun): the path has no inter-GPU step here ("replicas only"): every rank runs
the same workload on its own GPU, value = total DOF-updates / max-over-ranks time, scaling = weak.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dg_dof_updates_per_s"
UNIT = "DOF-updates/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2_two_layer")
    ap.add_argument("--timesteps", type=int, default=0, help="global time steps per bench step (0 = the config's)")
    ap.add_argument("--precision", type=int, default=0)
    ap.add_argument("--order", type=int, default=0)
    ap.add_argument("--hexes", default="", help="nx,ny,nz override (development)")
    ap.add_argument("--no-extras", action="store_true", help="skip cpu_baseline and the per-config extras")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# --------------------------------------------------------------------------------------------------
# algorithmic traffic per element and launch, in scalars
# --------------------------------------------------------------------------------------------------
def algorithmic_scalars(kernel, Np, Nfp):
    if kernel == "step":           # fused rhs + update: q in/out, nbr traces in, 2 rhs in, 1 rhs out, traces out
        return 20 * Np + 16 * Nfp + 31
    if kernel == "step_image":     # the same for two wavefields + image read-modify-write
        return 2 * (20 * Np + 16 * Nfp + 31) + 2 * Np
    if kernel == "rhs":            # unfused volume + surface: q in, neighbour traces in, factors, rhs out
        return 8 * Np + 8 * Nfp + 31
    if kernel == "update":         # q in/out, three right-hand sides in, exposed traces out
        return 20 * Np + 8 * Nfp
    if kernel == "image_update":   # two wavefields + image read-modify-write
        return 2 * (20 * Np + 8 * Nfp) + 2 * Np
    raise KeyError(kernel)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            parts = [x.strip() for x in r.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def build_workload(args):
    from workloads import make_config
    kw = {}
    if args.hexes:
        kw["hexes"] = tuple(int(x) for x in args.hexes.split(","))
    if args.order:
        kw["N"] = args.order
    if args.precision:
        kw["precision"] = args.precision
    cfg = make_config(args.workload, **kw)
    T = args.timesteps or cfg["nsteps"]
    return cfg, T


def dof_updates_per_global_step(levels, Np):
    """Sum over levels of K_l 2^level 4 Np (= 4 K Np when single-rate)."""
    cnt = np.bincount(levels)
    return int(sum(int(c) * (1 << l) for l, c in enumerate(cnt)) * 4 * Np)


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------
def make_ctx(cfg, device, history_steps=0):
    import paper_1506_00907_b200 as pk
    g = pk.DG(cfg["N"], cfg["precision"], cfg["EToV"], cfg["VX"], default_bc=cfg["default_bc"])
    g.dg_set_model(cfg["rho"], cfg["c"], cfg["nlevels"], cfg["cfl"])
    if cfg.get("source"):
        s = cfg["source"]
        g.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    if cfg.get("receivers") is not None and history_steps:
        g.dg_set_receivers(cfg["receivers"])
    g.bind_torch(device)
    if history_steps:
        g.bind_history_torch(history_steps, device)
    return g


def max_over_ranks(sec, dist, device):
    """Time of a multi-rank run = the slowest rank's device time (dist: an initialised torch.distributed)."""
    if dist is None:
        return sec
    import torch
    t = torch.tensor([sec], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(dof_per_rank_step, steps, world, sec):
    """Replicas only: every rank advances the same workload; value = all ranks' DOF-updates / slowest time."""
    return world * dof_per_rank_step * steps / sec


def timed_steps(g, torch, T, K, W, dist, device):
    """W warm-up + K timed bench steps of dg_step(T) on the bound stream; returns max-over-ranks seconds."""
    for _ in range(W):
        g.dg_step(T)
    torch.cuda.synchronize(device)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(device)
    n0 = g.dg_get_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        g.dg_step(T)
    e1.record()
    torch.cuda.synchronize(device)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(device)
    sec = max_over_ranks(e0.elapsed_time(e1) * 1e-3, dist, device)
    return sec, g.dg_get_launch_count() - n0


def profile_kernels(g, T, reps, elems_per_global_step, Np, Nfp, rs, peak, peak_src, ncu_traffic=None):
    """Separate pass with one event pair per launch: per-kernel average durations inside the step.
    achieved = algorithmic bytes of all launches of the class / their summed event time."""
    g.dg_step(min(T, 50))
    g.dg_get_kernel_times()
    g.dg_set_profiling(True)
    for _ in range(reps):
        g.dg_step(T)
    times = g.dg_get_kernel_times()
    g.dg_set_profiling(False)
    ker = {}
    for name in ("step", "step_image", "rhs", "update", "image_update"):
        ms, n = times[name]
        if not n:
            continue
        nbytes = float(reps) * T * elems_per_global_step * algorithmic_scalars(name, Np, Nfp) * rs
        gbs = nbytes / (ms * 1e-3) * 1e-9
        ker[name] = {"launches": n, "avg_us": round(ms * 1e3 / n, 3),
                     "algorithmic_bytes_per_launch": int(nbytes / n),
                     "achieved_gbs": round(gbs, 1), "frac": round(gbs / peak, 4)}
    total = sum(v[0] for v in times.values())
    other = total - sum(times[k][0] for k in ker)
    dom = max(ker, key=lambda k: times[k][0])
    roof = {"bound": "hbm", "kernel": dom, "achieved": ker[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
            "frac": ker[dom]["frac"], "traffic": ncu_traffic, "peak_source": peak_src,
            "share_of_step": round(times[dom][0] / total, 4) if total else None}
    return roof, ker, {"other_kernels_ms": round(other, 3), "all_kernels_ms": round(total, 3)}


def run_e2e(g, torch, T, K, q0, device):
    """Same metric through the C ABI with host buffers: set_state(host) -> step -> get_fields(host)."""
    g.dg_set_state(q0)
    g.dg_step(T)
    g.dg_get_fields()
    torch.cuda.synchronize(device)
    t0 = time.perf_counter()
    for _ in range(K):
        g.dg_set_state(q0)
        g.dg_step(T)
        q = g.dg_get_fields()
    torch.cuda.synchronize(device)
    sec = time.perf_counter() - t0
    return sec, q


# --------------------------------------------------------------------------------------------------
# the oracle on the host cores: cpu_baseline and --impl reference
# --------------------------------------------------------------------------------------------------
def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info()]
        return max(n) if n else 1
    except Exception:
        return 1


def make_oracle(cfg):
    from oracle.dgtd import DGOracle
    o = DGOracle(cfg["N"], cfg["EToV"], cfg["VX"], default_bc=cfg["default_bc"])
    o.set_model(cfg["rho"], cfg["c"], cfg["nlevels"], cfg["cfl"])
    if cfg.get("source"):
        s = cfg["source"]
        o.set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    return o


def time_oracle(o, F, nglobal, t0):
    t = time.perf_counter()
    o.run_mrab([F], nglobal, t0)
    return time.perf_counter() - t


def cpu_baseline(cfg, budget_s=15.0):
    """The oracle as it stands on a bounded sample: as many global time steps of the same workload as
    fit in about budget_s seconds (the rate does not depend on the step count)."""
    o = make_oracle(cfg)
    F = o.new_field()
    dt_g = o.dt_local * o.nlocal
    sec1 = time_oracle(o, F, 1, 0.0)
    n = int(max(1, min(50, budget_s / max(sec1, 1e-3))))
    sec = time_oracle(o, F, n, dt_g)
    dof = dof_updates_per_global_step(o.level, o.Np)
    return {"value": dof * n / sec, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
            "sample": "%d global time steps of %s (K=%d, N=%d, fp64 numpy), %.1f s" % (n, cfg["name"], o.K, cfg["N"], sec)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, T = build_workload(args)
    o = make_oracle(cfg)
    F = o.new_field()
    dt_g = o.dt_local * o.nlocal
    dof = dof_updates_per_global_step(o.level, o.Np)
    sec1 = time_oracle(o, F, 1, 0.0)                      # also the first warm-up
    # each step = a bounded sample: n global time steps so that the whole run stays within minutes
    total_budget = 120.0
    n = int(max(1, min(T, total_budget / max(sec1, 1e-3) / max(1, args.steps + args.warmup))))
    done = 1
    for _ in range(max(0, args.warmup - 1)):
        time_oracle(o, F, n, done * dt_g)
        done += n
    t = time.perf_counter()
    for _ in range(args.steps):
        o.run_mrab([F], n, done * dt_g)
        done += n
    sec = time.perf_counter() - t
    value = dof * n * args.steps / sec
    sample = "%d global time steps per step (of the config's %d) on %s K=%d N=%d" % (n, T, cfg["name"], o.K, cfg["N"])
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "K": int(o.K), "N": cfg["N"], "hexes": list(cfg["hexes"]),
                       "note": "the reference is a paper: this arm is the fp64 numpy oracle on the host cores"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
# extras (rank 0, N = 1): the other items of BASELINE.json's metric
# --------------------------------------------------------------------------------------------------
def extra_sweep(torch, device, peak, peak_src, hexes):
    """DOF-updates/s and per-kernel GB/s at N = 3, 4 in fp32 and fp64 on a mesh far larger than L2
    (config-4-sized jittered box, single-rate) and with the three LTS levels of config 3's grading."""
    from workloads import make_config
    out = []
    for name, N, prec, T in (("cfg4_rtm", 3, 32, 60), ("cfg4_rtm", 3, 64, 40), ("cfg4_rtm", 4, 32, 40),
                             ("cfg4_rtm", 4, 64, 30), ("cfg3_lts", 4, 32, 20), ("cfg3_lts", 3, 32, 20)):
        cfg = make_config(name, hexes=hexes.get(name), N=N, precision=prec)
        cfg["receivers"] = None
        g = make_ctx(cfg, device)
        levels = g.dg_get_levels()
        dof = dof_updates_per_global_step(levels, g.Np)
        sec, _ = timed_steps(g, torch, T, 3, 1, None, device)
        roof, ker, oth = profile_kernels(g, T, 1, dof // (4 * g.Np), g.Np, g.Nfp, prec // 8, peak, peak_src)
        out.append({"workload": name, "K": int(g.K), "N": N, "dtype": "f%d" % prec,
                    "levels": np.bincount(levels).tolist(), "value": dof * T * 3 / sec, "unit": UNIT,
                    "ms_per_global_time_step": 1e3 * sec / (3 * T), "kernels": ker, **oth})
        g.close()
        del g
        torch.cuda.empty_cache()
    return out


def extra_rtm_shot(torch, device, peak, peak_src, hexes, nsteps):
    """One full RTM shot of config 4 through the C ABI (host data buffers): forward with trace capture
    and receiver recording, backward with trace replay, receiver injection and fused imaging."""
    from workloads import make_config
    cfg = make_config("cfg4_rtm", hexes=hexes, nsteps=nsteps)
    nsteps = cfg["nsteps"]
    g = make_ctx(cfg, device, history_steps=nsteps)
    torch.cuda.synchronize(device)
    t0 = time.perf_counter()
    data = g.rtm_forward_shot(nsteps)
    t1 = time.perf_counter()
    g.rtm_backward_shot(nsteps, data, updir=tuple(cfg["updir"]))
    t2 = time.perf_counter()
    img = g.rtm_image_read()
    t3 = time.perf_counter()
    dof = 4 * g.K * g.Np
    # kernel shares of the backward phase (second, short pass with event pairs)
    g.dg_set_profiling(True)
    g.rtm_backward_shot(min(nsteps, 50), None, updir=tuple(cfg["updir"]))
    times = g.dg_get_kernel_times()
    g.dg_set_profiling(False)
    rs = cfg["precision"] // 8
    ker = {}
    nb = min(nsteps, 50)
    for name, fields in (("step_image", 1),):
        ms, n = times[name]
        if n:
            nbytes = float(nb) * fields * g.K * algorithmic_scalars(name, g.Np, g.Nfp) * rs
            ker[name] = {"launches": n, "avg_us": round(ms * 1e3 / n, 2), "achieved_gbs": round(nbytes / ms * 1e-6, 1),
                         "frac": round(nbytes / ms * 1e-6 / peak, 4)}
    out = {"workload": "cfg4_rtm", "K": int(g.K), "N": cfg["N"], "dtype": "f%d" % cfg["precision"], "nsteps": nsteps,
           "receivers": int(g.nr), "forward_s": t1 - t0, "backward_s": t2 - t1, "image_read_s": t3 - t2,
           "shot_s": t3 - t0, "forward_dof_updates_per_s": dof * nsteps / (t1 - t0),
           "backward_dof_updates_per_s": 2 * dof * nsteps / (t2 - t1),
           "history_gb": g.rtm_history_bytes(nsteps) * 1e-9, "image_l2": float(np.linalg.norm(img)),
           "backward_kernels": ker}
    g.close()
    return out


def run_ours(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the DGTD hot path has no CPU fallback)")
    device = "cuda:%d" % local
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist_mod.init_process_group("nccl", device_id=torch.device(device))
        dist = dist_mod
    peak, peak_src = load_peaks()
    cfg, T = build_workload(args)
    g = make_ctx(cfg, device)
    levels = g.dg_get_levels()
    Np, Nfp, rs = g.Np, g.Nfp, cfg["precision"] // 8
    dof_step = dof_updates_per_global_step(levels, Np)          # per global time step
    K, W = args.steps, max(args.warmup, 0)

    sampler = ClockSampler(local)
    sampler.start()
    sec, launches = timed_steps(g, torch, T, K, W, dist, device)
    clocks = sampler.stop()
    value = whole_job_value(dof_step * T, K, world, sec)

    # roofline of the dominant kernel: separate pass, one event pair per launch
    roof, ker, oth = profile_kernels(g, T, max(1, min(K, 3)), dof_step // (4 * Np), Np, Nfp, rs, peak, peak_src,
                                     ncu_traffic=NCU_TRAFFIC.get((cfg["name"], cfg["N"], cfg["precision"])))
    roof["timing"] = "one CUDA event pair per launch (dg_set_profiling), separate pass over the same steps"
    if len(ker) == 1 and oth["other_kernels_ms"] == 0.0 and launches == K * T * (1 << (cfg["nlevels"] - 1)):
        # the step is ONE kernel launched back to back: its average launch duration over the timed region is
        # the timed region / launches (the event pairs of the separate pass break the dependent-launch overlap)
        dom = roof["kernel"]
        avg_s = sec / launches
        nbytes = ker[dom]["algorithmic_bytes_per_launch"]
        roof["event_pair_pass"] = {"avg_us": ker[dom]["avg_us"], "achieved": roof["achieved"], "frac": roof["frac"]}
        roof["achieved"] = round(nbytes / avg_s * 1e-9, 1)
        roof["frac"] = round(nbytes / avg_s * 1e-9 / peak, 4)
        roof["avg_launch_us"] = round(avg_s * 1e6, 3)
        roof["timing"] = "CUDA events around the timed region / launches in it (the step is this one kernel)"

    # end to end through the C ABI with host buffers
    rng = np.random.default_rng(0)
    q0 = 1e-3 * rng.standard_normal((g.K, 4, Np))
    Ke = max(1, min(K, 5))
    sec_e, _ = run_e2e(g, torch, T, Ke, q0, device)
    sec_e = max_over_ranks(sec_e, dist, device)
    field_bytes = int(g.K) * 4 * Np * rs
    e2e = {"value": world * dof_step * T * Ke / sec_e, "unit": UNIT, "h2d_bytes_per_step": field_bytes,
           "d2h_bytes_per_step": field_bytes, "ms_per_step": 1e3 * sec_e / Ke,
           "call": "dg_set_state(host q) -> dg_step(%d) -> dg_get_fields(host q), pageable numpy buffers" % T}
    ws_bytes = g.dg_workspace_bytes()
    g.close()
    del g
    torch.cuda.empty_cache()

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": 1e3 * sec / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f%d" % cfg["precision"], "data": "synthetic",
            "config": {"workload": cfg["name"], "hexes": list(cfg["hexes"]), "K": int(cfg["EToV"].shape[0]),
                       "N": cfg["N"], "Np": Np, "levels": np.bincount(levels).tolist(),
                       "time_steps_per_step": T, "integrator": "ab3", "parallelism": "replicas x%d" % world,
                       "l2": "no flush: every time step streams the whole %.0f MB workspace (q, 3 rhs, traces, "
                             "factors) and a bench step is %d consecutive time steps" % (ws_bytes * 1e-6, T)},
            "roofline": roof, "kernels": ker, **oth, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "us_per_time_step": 1e6 * sec / (K * T)}
    if rank == 0 and world == 1 and not args.no_extras:
        line["cpu_baseline"] = cpu_baseline(cfg)
        big = args.workload == "cfg2_two_layer" and not args.hexes
        line["sweep_large_mesh"] = extra_sweep(torch, device, peak, peak_src,
                                               {} if big else {"cfg4_rtm": (8, 8, 4), "cfg3_lts": (8, 8, 8)})
        line["rtm_shot"] = extra_rtm_shot(torch, device, peak, peak_src, None if big else (8, 8, 4),
                                          None if big else 20)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed
# `ncu --set full` capture (profiles/), keyed by (workload, N, precision); None until captured
NCU_TRAFFIC = {("cfg2_two_layer", 3, 32): 199077632}      # profiles/r1b_fused_pipeline.md (148.27 MB read + 50.81 MB written)


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)

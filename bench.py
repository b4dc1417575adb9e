#!/usr/bin/env python
"""bench.py -- GLUPS of the fused TSLB sweep (BASELINE.json metric) on N B200s of one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 512] [--dtype f32] [--kernel auto|gather|tile]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

A "step" is one lattice time step = one pass of the whole hot path (boundary
fill where the boundary set has open faces, the ghost-layer refresh, the fused stream-collide sweep, the buffer swap) over the whole
lattice.  Workload: BASELINE.json configs[4], periodic cube n^3 (default 512^3 fp32, the case the metric's
>= 70 % bar is quoted on), seeded random-phase Taylor-Green init, tau = 0.501.  GLUPS = n^3 * K / (1e9 T)
(Eq. 28).  One JSON line on stdout (rank 0).

The path does not shard (replicas only): with --gpus N > 1 every rank advances its own
independent replica of the lattice, `value` is the sum over ranks divided by the slowest rank's time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

BYTES_PER_SITE = {"f32": 80, "f64": 160}     # 10 moments read + 10 written
FALLBACK_HBM_GBS = 6650.0                     # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=512, help="cube edge of the configs[4] workload")
    ap.add_argument("--workload", default="cube", choices=["cube", "channel", "jet"],
                    help="cube = configs[4] (the headline, edge --n); channel = configs[2] 384x128x192; jet = configs[3] 256x256x768")
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "gather", "tile"])
    ap.add_argument("--order", type=int, default=3, choices=[2, 3],
                    help="Hermite order of the reconstruction: 3 = the paper's high-order TSLB (the headline), 2 = Eq. 8")
    ap.add_argument("--slabs", type=int, default=0,
                    help="opt-in: ONE lattice cut into this many z slabs (paper_2401_17074_b200/slab.py) instead of replicas: "
                         "under torchrun one slab per rank (must equal the world size, NCCL point-to-point exchange, strong "
                         "scaling); on one GPU all slabs on it with device-copy exchange (cost of the decomposition path)")
    ap.add_argument("--staged", action="store_true",
                    help="with --slabs: ghost planes through tslb_export_face / tslb_import_face instead of in place (tslb_face_planes)")
    ap.add_argument("--connected", action="store_true",
                    help="with --slabs: no exchange at all, the tile kernel reads the neighbouring slabs' planes in place "
                         "(tslb_set_neighbor; under torchrun through CUDA IPC mappings of the neighbours' workspaces)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip timing the oracle on the host cores")
    ap.add_argument("--cpu-budget-s", type=float, default=15.0)
    return ap.parse_args(argv)


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
            t0 = time.time()                      # nvidia-smi needs a moment to start: wait for its first sample, so that even
            while not self.lines and time.time() - t0 < 2.0:   # a timed region shorter than the sampling period has a reading
                time.sleep(0.01)
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return None
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thr.join(timeout=5)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            p = [x.strip() for x in l.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
                try:
                    pw.append(float(p[2]))
                except ValueError:
                    pass
            except ValueError:
                continue
            for nme, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        if not sm:
            return None
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": max(mx), "power_w_max": max(pw) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# aggregation over ranks (also exercised on CPU with gloo, world_size 2: tests/test_bench_host.py)
# ------------------------------------------------------------------------------------------------
def aggregate(local_ms: float, local_units: float, dist=None, device="cpu"):
    """(max over ranks of the elapsed ms, sum over ranks of the units processed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def glups(units: float, ms: float) -> float:
    return units / (ms * 1e-3) / 1e9


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload_key: str):
    """DRAM bytes per launch of the sweep kernel from the committed ncu --set full summary, or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(workload_key)
    except Exception:
        return None


# ------------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline of our line; the whole of --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sample(w, edge: int):
    """Periodic sub-cube [0, edge)^3 cut from the workload's initial state: a bounded sample of it."""
    import numpy as np
    return np.ascontiguousarray(w.moments[:, :edge, :edge, :edge])


def time_oracle(w, edge: int, steps: int, warmup: int):
    import oracle                     # test infrastructure; allowed here (cpu_baseline / --impl reference only)
    M = oracle_sample(w, edge)
    o = oracle.Oracle(edge, edge, edge, w.tau)
    o.set_moments(M)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    return dt, oracle.num_threads()


def cpu_baseline(w, budget_s: float):
    edge = min(128, w.nx, w.ny, w.nz)
    dt1, cores = time_oracle(w, edge, 1, 0)
    steps = max(2, min(50, int(budget_s / max(dt1, 1e-6))))
    dt, cores = time_oracle(w, edge, steps, 0)
    return {"value": edge**3 * steps / dt / 1e9, "unit": "GLUPS", "cores": cores, "kind": "oracle",
            "sample": "%d steps of the fp64 oracle on the %d^3 periodic sub-cube [0,%d)^3 of the same initial state"
                      % (steps, edge, edge)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2401_17074_b200 import workloads as W
    edge = min(64, args.n)
    if args.workload == "cube":
        w = W.throughput(args.n, args.dtype, args.steps, edge=edge)     # the sub-cube [0,edge)^3 of the same field
    else:
        w = make_workload(args)
    dt, cores = time_oracle(w, edge, args.steps, args.warmup)
    val = edge**3 * args.steps / dt / 1e9
    sample = ("each step = one fp64 oracle sweep of a %d^3 periodic sub-cube of the configs[4] initial state "
              "(bounded sample of the %d^3 workload)" % (edge, args.n))
    line = {"impl": "reference", "metric": "GLUPS", "value": val, "unit": "GLUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args),
            "cpu_baseline": {"value": val, "unit": "GLUPS", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def make_workload(args):
    from paper_2401_17074_b200 import workloads as W
    if args.workload == "channel":
        return W.channel(steps=args.steps, dtype=args.dtype)
    if args.workload == "jet":
        return W.jet(steps=args.steps, dtype=args.dtype)
    return W.throughput(args.n, args.dtype, args.steps)


def workload_config(args):
    es = 4 if args.dtype == "f32" else 8
    if args.workload == "channel":
        what, sites = ("BASELINE.json configs[2]: D3Q27 TSLB channel 384x128x192 %s, halfway bounce-back walls in y, body force, "
                       "laminar parabola + seeded 5%% perturbation" % args.dtype), 384 * 128 * 192
    elif args.workload == "jet":
        what, sites = ("BASELINE.json configs[3]: D3Q27 TSLB jet 256x256x768 %s, velocity inlet (disc D=20, 1%% seeded noise) at z=0, "
                       "zero-gradient outlets elsewhere" % args.dtype), 256 * 256 * 768
    else:
        what, sites = ("BASELINE.json configs[4]: D3Q27 TSLB periodic cube %d^3 %s, random-phase Taylor-Green "
                       "U0=0.02 (seed=%d), tau=0.501" % (args.n, args.dtype, args.n)), args.n**3
    return {"workload": what, "sites": sites,
            "l2": "inputs larger than L2 (state %.2f GB vs 126 MB)" % (2 * 10 * sites * es / 1e9),
            "parallelism": "replicas x%d (path does not shard)" % args.gpus}


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2401_17074_b200 import binding as B
    from paper_2401_17074_b200 import build as BLD
    from paper_2401_17074_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the TSLB path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    BLD.build_lib()
    kernel = {"auto": B.KERNEL_AUTO, "gather": B.KERNEL_GATHER, "tile": B.KERNEL_TILE}[args.kernel]

    w = make_workload(args)
    w.order = args.order
    sim = B.from_workload(w, kernel)
    host = torch.from_numpy(w.moments)
    sim.set_moments(host.to("cuda"))
    stream = torch.cuda.current_stream()
    kname = B.KERNEL_NAMES[sim.active_kernel()]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg ---------------------------------------------------------------
    sim.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    l0 = sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    sim.step(args.steps)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count - l0
    clocks = sampler.stop() if rank == 0 else None
    ms_max, units = aggregate(ms, float(w.sites) * args.steps, dist if world > 1 else None, "cuda")
    value = glups(units, ms_max)

    # ---- the sweep kernel alone: event pairs around every sweep launch, outside the timed region ---------
    nt = max(1, min(args.steps, 50))
    sim.set_timing(nt)
    sim.step(nt)
    torch.cuda.synchronize()
    sweep_n, sweep_tot = sim.get_timing()
    sim.set_timing(0)
    sweep_ms = sweep_tot / max(sweep_n, 1)

    # sanity: the state is finite and mass is conserved (periodic box) -- not part of the timed region
    d = sim.diagnostics().cpu().numpy()
    assert np.isfinite(d).all() and (args.workload == "jet" or abs(d[0] / w.sites - 1) < 1e-5), d

    # ---- end-to-end leg: host buffers through the C ABI, copies inside the timed region -----
    e2e = None
    if not args.no_e2e:
        pinned = torch.empty(host.shape, dtype=host.dtype, pin_memory=True)
        pinned.copy_(host)
        barrier()
        t0 = time.perf_counter()
        e0.record(stream)
        sim.set_moments_host(pinned)             # H2D of the initial state
        sim.step(args.steps)
        sim.get_moments_host(pinned)             # D2H of the result (synchronises)
        e1.record(stream)
        barrier()
        ms_e = max(e0.elapsed_time(e1), 0.0)
        ms_e_max, units_e = aggregate(ms_e, float(w.sites) * args.steps, dist if world > 1 else None, "cuda")
        nbytes = host.numel() * host.element_size()
        e2e = {"value": glups(units_e, ms_e_max), "unit": "GLUPS",
               "h2d_bytes_per_step": nbytes / args.steps, "d2h_bytes_per_step": nbytes / args.steps,
               "what": "tslb_set_moments_host (pinned) + tslb_step(%d) + tslb_get_moments_host, whole job; "
                       "bytes are the one-off state copies amortised over the steps" % args.steps,
               "wall_s": time.perf_counter() - t0}
        assert np.isfinite(pinned.numpy()[:, ::64, ::64, ::64]).all()
        del pinned

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_src = hbm_peak()
    # Dominant kernel = the sweep.  When the timed region holds exactly one launch per step (periodic / wall runs: the
    # sweep keeps the ghost layers current itself) its average duration is taken over the timed region itself; otherwise
    # from the event pairs around the sweep launches of the extra pass.
    one_per_step = launches == args.steps
    kernel_ms = ms / args.steps if one_per_step else sweep_ms
    achieved = BYTES_PER_SITE[args.dtype] * w.sites / (kernel_ms * 1e-3) / 1e9
    roof = {"bound": "hbm", "kernel": "sweep_%s_kernel<%s>" % (kname, args.dtype), "achieved": achieved, "peak": peak,
            "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
            "algorithmic_bytes_per_site": BYTES_PER_SITE[args.dtype],
            "kernel_ms": kernel_ms, "kernel_share_of_step": kernel_ms / (ms / args.steps),
            "how": ("CUDA events around the timed region, %d sweep launches = %d steps" % (launches, args.steps)) if one_per_step
                   else ("CUDA event pairs around each sweep launch (tslb_set_timing), %d steps run after the timed region" % sweep_n),
            "kernel_ms_event_pairs": sweep_ms, "kernel_launches_event_pairs": sweep_n,
            "traffic": ncu_traffic("%s_%s_%s" % (kname, args.n if args.workload == "cube" else args.workload, args.dtype))}
    line = {"metric": "GLUPS", "value": value, "unit": "GLUPS", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": args.dtype, "data": "synthetic", "config": dict(workload_config(args), kernel=kname, order=args.order),
            "roofline": roof, "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches)}
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(w, args.cpu_budget_s)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_slabs(args):
    """--slabs S: the same workload as one lattice cut into S slabs along z.  Not the default: the
    north_star's path is one GPU / replicas; this leg measures what the decomposition costs."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2401_17074_b200 import binding as B
    from paper_2401_17074_b200 import build as BLD
    from paper_2401_17074_b200 import slab as S
    from paper_2401_17074_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the TSLB path has no CPU fallback")
    if world > 1 and args.slabs != world:
        raise SystemExit("bench.py: --slabs must equal the world size under torchrun (one slab per rank)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    BLD.build_lib()
    kernel = {"auto": B.KERNEL_AUTO, "gather": B.KERNEL_GATHER, "tile": B.KERNEL_TILE}[args.kernel]
    w = make_workload(args)
    w.order = args.order
    plans = S.plan_slabs(w.nz, args.slabs, w.faces.get(W.FACE_ZLO, W.BC_PERIODIC) == W.BC_PERIODIC)
    slabs = [S.Slab(w, p, kernel, args.staged, ipc=args.connected and world > 1) for p in (plans if world == 1 else [plans[rank]])]
    owned_sites = float(sum(s.plan.owned for s in slabs)) * w.nx * w.ny
    stream = torch.cuda.current_stream()

    if args.connected:
        if world > 1:
            S.connect_ipc(slabs[0])         # the neighbours' workspaces mapped through CUDA IPC (NVLink peer memory)
        else:
            S.connect_local(slabs)

    def advance(n):
        if world > 1 and args.connected:
            S.step_connected_dist(slabs[0], n)
        elif world > 1:
            slabs[0].step(n)
        elif args.connected:
            S.step_connected(slabs, n)
        else:
            S.step_local(slabs, n)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    advance(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    l0 = sum(s.sim.launch_count for s in slabs)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    advance(args.steps)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = sum(s.sim.launch_count for s in slabs) - l0
    clocks = sampler.stop() if rank == 0 else None
    ms_max, units = aggregate(ms, owned_sites * args.steps, dist if world > 1 else None, "cuda")
    d = sum(s.diagnostics(reduce=False) for s in slabs)
    if world > 1:
        dist.all_reduce(d)
    d = d.cpu().numpy()
    assert np.isfinite(d).all() and (args.workload == "jet" or abs(d[0] / w.sites - 1) < 1e-5), d
    # the sweeps alone (event pairs around each sweep launch of every local slab), after the timed region
    nt = max(1, min(args.steps, 20))
    for s in slabs:
        s.sim.set_timing(nt)
    advance(nt)
    torch.cuda.synchronize()
    sweep_ms = sum(s.sim.get_timing()[1] for s in slabs) / nt
    for s in slabs:
        s.sim.set_timing(0)
    if rank == 0:
        peak, peak_src = hbm_peak()
        step_ms = ms_max / args.steps
        achieved = BYTES_PER_SITE[args.dtype] * (units / args.steps) / (step_ms * 1e-3) / 1e9
        cfg = dict(workload_config(args), order=args.order, kernel=B.KERNEL_NAMES[slabs[0].sim.active_kernel()])
        cfg["parallelism"] = ("one lattice in %d z slabs, " % args.slabs) + (
            ("one slab per GPU, " + ("neighbours' planes read over CUDA IPC peer memory, one NCCL all-reduce per step as barrier"
                                     if args.connected else "ghost planes by NCCL point-to-point")) if world > 1 else
            "all on one GPU, " + ("no exchange" if args.connected else "ghost planes by device copies"))
        cfg["slab_planes"] = [p.owned for p in plans]
        cfg["transport"] = ("none: neighbours read in place by the sweep's TMA producer (tslb_set_neighbor)" if args.connected else
                            "staged (tslb_export_face / tslb_import_face)" if args.staged else "in place (tslb_face_planes)")
        line = {"metric": "GLUPS", "value": glups(units, ms_max), "unit": "GLUPS", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": args.dtype, "data": "synthetic", "config": cfg,
                "roofline": {"bound": "hbm", "kernel": "whole step: sweep of every local slab + face export / transport / import",
                             "achieved": achieved, "peak": (peak * world) if peak else None, "unit": "GB/s",
                             "frac": achieved / (peak * world) if peak else None, "peak_source": peak_src,
                             "algorithmic_bytes_per_site": BYTES_PER_SITE[args.dtype], "traffic": None,
                             "sweep_ms_per_step_rank0": sweep_ms, "exchange_ms_per_step_rank0": ms / args.steps - sweep_ms},
                "clocks": clocks, "e2e": None, "gpu_launches": int(launches)}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    args = parse_args(argv)
    if args.impl == "reference":
        return run_reference(args)
    if args.slabs > 1:
        return run_slabs(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

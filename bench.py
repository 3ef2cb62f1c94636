#!/usr/bin/env python
"""bench.py -- zones burned/sec on the 13-isotope 128^3 config (BASELINE.json configs[2]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]
                    [--static-schedule] [--kernel auto|coop|quad] [--order cost|index|steps]

A "step" is one pass of the whole hot path (a1-a9: load, work queue, rates, Jacobian, LU,
Newton, BDF control, store) over one batch of synthetic zones: one burn_zones call.
N > 1: one process per GPU, every rank burns its own copy of the config (weak scaling, no data-path
collective); value = zones of all ranks / max time.  Started under torchrun the
ranks are used as given; started plainly with --gpus N > 1 the script re-launches itself under
torch.distributed.run with N ranks on 127.0.0.1.
Prints ONE JSON line on rank 0.  DESIGN.md section 6 defines every field.
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

from workloads import CONFIG_NZ, make_workload  # noqa: E402

METRIC = "zones burned/sec (13-isotope net, fp64 BDF)"
UNIT = "zones/s"
FP64_LANES_PER_SM = 64           # DFMA lanes per SM
CPU_SAMPLE_STRIDE = {1: 1, 2: 16, 3: 64, 4: 64, 5: 512}
SINGLE_CORE_STRIDE = {1: 1, 2: 128, 3: 1024, 4: 8192, 5: 4096}   # <= 4096 zones, one thread (the axis of PAPER.md:L127 Fig. 5)


def _workload_name(cfg):
    return {1: "config1 carbon 3-ODE 4096 zones", 2: "config2 alpha7 64^3", 3: "config3 alpha13 128^3 XRB-like",
            4: "config4 alpha13 256^3 hotspots", 5: "config5 synth30 128^3"}[cfg]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows = []
        self.proc = None
        self.gpu = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 9 for n, v in zip(names, r[5:9]) if v.lower().startswith("active")})
        pw = [float(r[3]) for r in self.rows if len(r) >= 9 and r[3].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores, on a bounded sample of the
    same workload (every s-th zone).  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    stride = CPU_SAMPLE_STRIDE[args.config]
    w = make_workload(args.config, zones=stride if stride > 1 else None)
    cores = oracle.max_threads()
    for _ in range(args.warmup):
        oracle.burn(w.net, w.rho[:256], w.T[:256], w.X[:, :256], w.dt, w.rtol, w.atol)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol)
    el = (time.perf_counter() - t0) / args.steps
    value = w.nz / el
    sample = f"every {stride}th zone of {_workload_name(args.config)} ({w.nz} zones per step)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": el * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_name(args.config), "zones_per_step": w.nz, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def _max_over_ranks(values, device, world):
    """Timings are reported as the MAX over ranks (the job is done when its slowest rank is)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def run_stub(args):
    """--stub (tests only, tests/test_bench_launcher.py): the multi-rank plumbing of run_ours --
    rendezvous, barrier, max-over-ranks timing, one JSON line from rank 0 -- with the gloo backend and a
    sleep in place of the burn, so that the N > 1 path can be exercised on a box without GPUs."""
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    nz = 1000
    for _ in range(args.warmup):
        time.sleep(0.001)
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time.sleep(0.01 * (rank + 1))            # rank r is (r + 1) x slower: the max must win
    total_ms = (time.perf_counter() - t0) * 1e3
    if world > 1:
        dist.barrier()
    (total_ms,) = _max_over_ranks([total_ms], torch.device("cpu"), world)
    if rank == 0:
        ms = total_ms / args.steps
        print(json.dumps({"metric": METRIC, "value": world * nz / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "stub": True,
                          "scaling": "weak", "config": {"workload": "stub (sleep)", "zones_per_gpu": nz}}))
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1711_06203_b200 as bz
    from paper_1711_06203_b200.flops import algorithmic_flops, flop_model, state_bytes_per_zone

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the burn has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = args.config
    # every rank burns its own full copy (weak scaling); --stride S (profiling only) = every S-th zone
    w = make_workload(cfg, zones=args.stride if args.stride > 1 else None)
    nz, N = w.nz, w.net.nspec
    net = bz.net_create(w.net)
    net.select_kernel(args.kernel)
    net.set_schedule("static" if args.static_schedule else ("cost" if args.order == "cost" else "queue"))
    net.set_policy(args.policy)
    stream = torch.cuda.current_stream()
    order_note = "zone index (bz_set_schedule 0)"
    if args.order == "cost" and not args.static_schedule:
        # the library's default: its own a-priori key, key kernel + radix sort INSIDE every timed burn
        order_note = ("by decreasing a-priori cost key |dT/dt| / T at the initial state (bz_set_schedule 2, the default: "
                      "one right-hand side per zone and a radix sort, inside the timed burn)")

    # ---- device-resident arm -------------------------------------------------------------------
    rho_d, T_d, X_d = (torch.from_numpy(a).to(dev) for a in (w.rho, w.T, w.X))
    To_d, Xo_d = torch.empty_like(T_d), torch.empty_like(X_d)
    ns_d = torch.empty(nz, dtype=torch.int32, device=dev)

    def step():
        bz.burn_zones(net, rho_d, T_d, X_d, w.dt, w.rtol, w.atol, T_out=To_d, X_out=Xo_d, nsteps=ns_d, stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.order == "steps":
        # a caller's order (bz_set_zone_order): by decreasing step count of a PREVIOUS burn of this batch -- what an
        # application that burns every hydro step knows from the step before; on a repeated identical batch it is
        # the ideal key.  Results do not depend on it.
        step()
        torch.cuda.synchronize()
        net.set_zone_order(torch.argsort(ns_d.to(torch.int64), descending=True, stable=True))
        order_note = "by decreasing step count of a previous burn of the same batch (a caller's order; ideal cost key)"

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for i in range(args.steps):
        step()
        ev[i + 1].record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    per_launch_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[-1])
    counters = bz.get_counters(net)              # of the last launch
    nfail = int((ns_d < 0).sum().item())

    # ---- end-to-end arm: host buffers through the C ABI, copies inside the timed region --------
    net.set_zone_order(None)   # (the host path burns in chunks and takes no caller's order)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    rho_h, T_h, X_h = pin(w.rho), pin(w.T), pin(w.X)
    To_h = torch.empty(nz, dtype=torch.float64).pin_memory()
    Xo_h = torch.empty((N, nz), dtype=torch.float64).pin_memory()
    ns_h = torch.empty(nz, dtype=torch.int32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))
    bz.burn_zones_host(net, rho_h, T_h, X_h, w.dt, w.rtol, w.atol, To_h, Xo_h, ns_h, stream=stream)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(e2e_steps):
        bz.burn_zones_host(net, rho_h, T_h, X_h, w.dt, w.rtol, w.atol, To_h, Xo_h, ns_h, stream=stream)
    e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1) / e2e_steps
    same = bool(np.array_equal(Xo_h.numpy(), Xo_d.cpu().numpy()))

    # ---- max over ranks ------------------------------------------------------------------------
    total_ms, e2e_ms = _max_over_ranks([total_ms, e2e_ms], dev, world)
    ms_per_step = total_ms / args.steps
    value = world * nz / (ms_per_step * 1e-3)
    e2e_value = world * nz / (e2e_ms * 1e-3)

    if rank == 0:
        # roofline of the dominant (only) kernel: plain FP64 ALUs
        props = torch.cuda.get_device_properties(dev)
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
        peak_tf = props.multi_processor_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        probe_tf, _ = bz.fp64_peak_probe(20000)
        aflops = algorithmic_flops(w.net, counters)
        kern_ms = float(np.mean(per_launch_ms))
        achieved = aflops / (kern_ms * 1e-3) / 1e12
        sbytes = state_bytes_per_zone(N)
        # two figures that only a profiler can give are COPIED from the committed ncu summaries of this
        # kernel on this config (profiles/ncu_counters.json names the capture); null when none exists
        traffic = executed = None
        ncu_src = None
        tpath = os.path.join(ROOT, "profiles", "ncu_counters.json")
        if os.path.exists(tpath):
            rec = json.load(open(tpath)).get(f"config{cfg}:{net.kernel_name}")
            if rec and not args.static_schedule and args.policy == "fresh" and args.order == "cost":
                traffic, executed, ncu_src = rec.get("dram_bytes"), rec.get("executed_fp64_flops"), rec.get("source")
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(cfg) + (f", every {args.stride}th zone" if args.stride > 1 else ""),
                       "zones_per_gpu": nz, "neq": N + 1, "nreac": w.net.nreac,
                       "dt": w.dt, "rtol": w.rtol, "atol": w.atol, "kernel": net.kernel_name,
                       "schedule": "static round-robin (a2 off)" if args.static_schedule else "work queue (a2)",
                       "queue_order": order_note,
                       "newton_matrix": "fresh J + LU every attempt (BZ-BDF v1)" if args.policy == "fresh"
                                        else "reused, VODE-style (BZ-BDF v2, DESIGN.md 12)",
                       "l2": (f"inputs {8 * (N + 2) * nz / 1e6:.0f} MB per step exceed the 126 MB L2" if 8 * (N + 2) * nz > 126e6
                              else f"inputs {8 * (N + 2) * nz / 1e6:.1f} MB per step fit the L2; the kernel is ALU-bound, "
                                   "state traffic is < 1e-3 of its time"),
                       "parallelism": f"zones sharded, {world} replica(s), no collective"},
            "rhs_evals_per_s": world * counters["nrhs"] / (kern_ms * 1e-3),
            "steps_per_zone_mean": counters["nst"] / nz, "failed_zones": nfail, "counters": counters,
            "hbm_state_gbs": sbytes * nz / (kern_ms * 1e-3) / 1e9,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s",
                         "frac": achieved / peak_tf, "traffic": traffic,
                         "traffic_source": ncu_src,
                         # FP64 flops the kernel EXECUTES per launch (ncu dadd + dmul + 2 dfma thread instructions,
                         # same capture) over the live kernel time: redundant lanes included, unlike `frac`
                         "executed_frac": (executed / (kern_ms * 1e-3) / 1e12 / peak_tf) if executed else None,
                         "peak_source": f"{props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x "
                                        f"{sm_max_mhz:.0f} MHz (derived); DFMA probe measured {probe_tf:.2f} TFLOP/s",
                         "frac_of_measured_probe": achieved / probe_tf,
                         "algorithmic_flops_per_launch": aflops, "kernel_ms": kern_ms,
                         "flop_model": flop_model(w.net)},
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms,
                    "h2d_bytes_per_step": 8 * (N + 2) * nz, "d2h_bytes_per_step": (8 * (N + 1) + 4) * nz,
                    "matches_device_path": same},
            # kernels of this repository inside the timed region: the burn kernel, and with the cost schedule the
            # key kernel before it (the radix sort between them is CUB's: 3-4 library kernels per step, not counted)
            "gpu_launches": args.steps * (2 if (args.order == "cost" and not args.static_schedule) else 1), "clocks": clocks,
        }
        if not args.no_cpu_baseline and world == 1:
            import oracle
            pol = 1 if args.policy == "reuse" else 0
            stride = CPU_SAMPLE_STRIDE[cfg]
            ws = make_workload(cfg, zones=stride if stride > 1 else None)
            t0 = time.perf_counter()
            oracle.burn(ws.net, ws.rho, ws.T, ws.X, ws.dt, ws.rtol, ws.atol, policy=pol)
            el = time.perf_counter() - t0
            out["cpu_baseline"] = {"value": ws.nz / el, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                                   "sample": f"every {stride}th zone ({ws.nz} zones), {el:.1f} s wall"}
            s1 = SINGLE_CORE_STRIDE[cfg]
            w1 = make_workload(cfg, zones=s1 if s1 > 1 else None)
            t0 = time.perf_counter()
            oracle.burn(w1.net, w1.rho, w1.T, w1.X, w1.dt, w1.rtol, w1.atol, nthreads=1, policy=pol)
            el1 = time.perf_counter() - t0
            out["cpu_baseline"]["single_core"] = {"value": w1.nz / el1, "unit": UNIT, "cores": 1,
                                                  "sample": f"every {s1}th zone ({w1.nz} zones), {el1:.1f} s wall"}
        print(json.dumps(out))
    bz.net_destroy(net)
    if world > 1:
        dist.destroy_process_group()


def relaunch(n, argv, extra_env=None):
    """`python bench.py --gpus N` without torchrun: start N ranks of this script on this node
    (one per GPU, rendezvous on 127.0.0.1) and hand their exit code back."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "WARN")
    env.update(extra_env or {})
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel", default="auto", choices=["auto", "coop", "quad"],
                    help="auto = specialised quad kernel when the topology has one, else the generic coop kernel")
    ap.add_argument("--order", default="cost", choices=["cost", "index", "steps"],
                    help="order in which the work queue hands the zones out: the library's a-priori cost key (default, "
                         "bz_set_schedule 2), zone index (bz_set_schedule 0), or decreasing step count of a previous "
                         "burn of the batch (bz_set_zone_order; device-resident arm only)")
    ap.add_argument("--static-schedule", action="store_true",
                    help="switch the work queue (step a2) off: static round-robin zone assignment, for the before/after figure")
    ap.add_argument("--policy", default="fresh", choices=["fresh", "reuse"],
                    help="Newton matrix: fresh J + LU on every attempt (default, the parity reference) or VODE-style reuse")
    ap.add_argument("--stride", type=int, default=1,
                    help="burn every S-th zone of the config only (short ncu captures; not a bench value)")
    ap.add_argument("--stub", action="store_true", help=argparse.SUPPRESS)   # tests only: see run_stub
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    world = os.environ.get("WORLD_SIZE")
    if world is None and args.gpus > 1:
        sys.exit(relaunch(args.gpus, sys.argv[1:]))
    if world is not None and int(world) != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with --nproc-per-node {args.gpus}")
    if args.stub:
        run_stub(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

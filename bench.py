#!/usr/bin/env python
"""bench.py -- site updates/s of one Swendsen-Wang step (arXiv 1403.7560) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

Prints ONE JSON line (rank 0).  A "step" is one pass of the whole hot path (bond activation ->
cluster labelling -> flip + magnetisation) over the configuration named in
`config.workload`; default C4 = 3D Ising L=512 at T=4.5115, the configuration BASELINE.json quotes
its HBM-roofline target on.  Inputs are synthetic and seed-defined (the simulation's own seeded
random start, thermalised by an untimed burn-in).  See DESIGN.md section 7 for every number's
definition.  `--impl reference` times the CPU oracle (oracle/), as it stands, on the host cores.
"""
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

METRIC = "site updates/sec per SW step"
UNIT = "site updates/s"
KERNELS = ("k_bond_label", "k_merge", "k_flip")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--burn-in", type=int, default=-1, help="untimed thermalisation steps (default per config)")
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--no-extras", action="store_true", help="skip cpu_baseline, e2e and the other configs")
    return ap.parse_args()


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def spin_bytes(model):
    return 4 if model == 2 else (2 if model == 3 else 1)


def floor_bytes_per_site(model):
    """spins read once and written once, a 4-byte label written before and
    read after the grid-wide merge; XY re-reads theta in the flip."""
    return 20 if model == 2 else (14 if model == 3 else 10)   # clock: uint16 states, re-read in the flip


def kernel_bytes_per_site(model):
    """Algorithmic bytes per site of each kernel."""
    sp = spin_bytes(model)
    return {"k_bond_label": sp + 4, "k_merge": 0, "k_flip": 4 + sp + (sp if model in (2, 3) else 0)}


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the one
# `ncu --set full` capture summarised in profiles/r01_final_ncu_full_C4.md (config -> kernel -> bytes).
NCU_TRAFFIC = {"C4": {"k_bond_label": 134.7e6 + 630.1e6, "k_merge": 380.1e6 + 74.6e6, "k_flip": 537.9e6 + 119.8e6}}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.samples, self._stop, self._thr = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 6:
                    self.samples.append(f)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        self._thr.join(timeout=10)

    def summary(self):
        sm = sorted(int(float(s[0])) for s in self.samples if s[0].replace(".", "").isdigit())
        mx = [int(float(s[1])) for s in self.samples if s[1].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({n for s in self.samples for n, v in zip(names, s[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.samples)}


def load_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
DEFAULT_BURN_IN = {"C1": 200, "C2": 200, "C3": 200, "C4": 150, "C5": 100, "X1": 100, "X2": 100, "X3": 100}
L2_BYTES = 126 * 2 ** 20


def working_set_bytes(cfg):
    n = cfg["L"] ** cfg["dim"]
    return n * (spin_bytes(cfg["model"]) + 1 + 4)


def time_config(sw, torch, cfg, seed, burn_in, warmup, steps, flush_buf):
    """Thermalise, warm up, then time `steps` SW steps with CUDA events (device time).
    Returns (context, ms_per_step, per-kernel ms list, launches)."""
    g = sw.SwendsenWang(cfg["dim"], cfg["L"], cfg["model"], cfg["q"], 1.0 / cfg["T"], seed=seed)
    g.step(burn_in)
    g.step(warmup)
    torch.cuda.synchronize()
    needs_flush = working_set_bytes(cfg) < 2 * L2_BYTES
    if not needs_flush:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.step(steps)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
    else:
        # working set comparable to L2: flush L2 (write a 512 MiB buffer) between timed steps
        tot = 0.0
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            flush_buf.add_(1)
            a.record()
            g.step(1)
            b.record()
        torch.cuda.synchronize()
        tot = sum(a.elapsed_time(b) for a, b in evs)
        ms = tot / steps
    # second pass over the same number of steps: per-kernel events (shares of the step)
    g.set_kernel_timing(True)
    for _ in range(steps):
        if needs_flush:
            flush_buf.add_(1)
        g.step(1)
    kms, ksteps = g.kernel_times()
    g.set_kernel_timing(False)
    kms = [x / max(ksteps, 1) for x in kms]
    return g, ms, kms, needs_flush


def measure_e2e(sw, torch, g, cfg, steps):
    """Same metric through the C ABI with HOST buffers: every step uploads the configuration from
    pinned host memory (sw_set_spins), runs one SW step, reads the observables and downloads the new
    configuration (sw_get_spins)."""
    n = g.N
    nbytes = n * spin_bytes(cfg["model"])
    host = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    g.get_spins_ptr(host.data_ptr(), nbytes)
    t = g.t
    for _ in range(2):
        g.set_spins_ptr(host.data_ptr(), nbytes, t)
        g.step(1)
        g.observables()
        g.get_spins_ptr(host.data_ptr(), nbytes)
        t += 1
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        g.set_spins_ptr(host.data_ptr(), nbytes, t)
        g.step(1)
        g.observables()
        g.get_spins_ptr(host.data_ptr(), nbytes)
        t += 1
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    return {"value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes + 2104,
            "what": "per step: sw_set_spins (pinned host -> device), sw_step(1), sw_observables, sw_get_spins (device -> pinned host)"}


def oracle_baseline(cfg, spins, t, max_seconds=30.0):
    """The CPU oracle, as it stands, on a bounded sample of the same workload: whole-lattice steps
    from the GPU's thermalised configuration, one thread."""
    from oracle import sw_oracle as orc
    o = orc.Oracle(cfg["dim"], cfg["L"], cfg["model"], cfg["q"], 1.0 / cfg["T"], 1)
    o.set_spins(spins, t)
    n = o.N
    done, t0 = 0, time.perf_counter()
    while True:
        o.step(1)
        done += 1
        el = time.perf_counter() - t0
        if el + el / done > max_seconds or done >= 1000:
            break
    o.close()
    return {"value": n * done / el, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{done} whole-lattice oracle step(s) of {cfg['desc']} from the GPU's thermalised state, "
                      f"{el:.1f} s on 1 thread of {os.cpu_count()} host cores", "ns_per_site": 1e9 * el / (n * done)}


def max_over_ranks(ms, device):
    """Replicas only: the job's step time is the slowest rank's; the one
    collective of the multi-GPU path (not on the data path).  Works on NCCL (cuda) and gloo (cpu)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1403_7560_b200 as sw
    from paper_1403_7560_b200 import inputs
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SW path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = {**inputs.CONFIGS, **inputs.EXTRA_CONFIGS}[args.config]
    n_sites = cfg["L"] ** cfg["dim"]
    burn = args.burn_in if args.burn_in >= 0 else DEFAULT_BURN_IN[args.config]
    warm = max(args.warmup, 3)
    flush_buf = torch.zeros(512 * 2 ** 20, dtype=torch.uint8, device="cuda")
    peak, peak_src = load_peak()

    # replicas only: every rank runs its own chain (seed + rank), no collective
    # on the data path; barrier + device timing, max over ranks.
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    with ClockSampler(local) as clk:
        g, ms, kms, flushed = time_config(sw, torch, cfg, args.seed + rank, burn, warm, args.steps, flush_buf)
    if world > 1:
        ms_all = max_over_ranks(ms, "cuda")
    else:
        ms_all = ms
    value = world * n_sites / (ms_all * 1e-3)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_all, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {0: "int8", 1: "u8", 2: "f32", 3: "u16"}[cfg["model"]], "data": "synthetic",
        "config": {"workload": f"{args.config}: {cfg['desc']} periodic, T={cfg['T']:.6f}, Philox seed {args.seed}"
                               f" (+rank), seeded random start thermalised by {burn} untimed SW steps",
                   "sites": n_sites, "burn_in_steps": burn,
                   "l2": "L2 flushed (512 MiB write) between timed steps" if flushed else "inputs larger than L2 (no flush)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "gpu_launches": 3 * args.steps,
        "clocks": clk.summary(),
    }
    # roofline of the dominant kernel: algorithmic bytes / CUDA-event duration / measured copy peak
    kb = kernel_bytes_per_site(cfg["model"])
    dom = max(range(3), key=lambda k: kms[k])
    name = KERNELS[dom]
    achieved = kb[name] * n_sites / (kms[dom] * 1e-3) / 1e9 if kms[dom] > 0 else 0.0
    step_gbs = floor_bytes_per_site(cfg["model"]) * n_sites / (ms * 1e-3) / 1e9
    out["roofline"] = {"bound": "hbm", "kernel": name, "achieved": achieved, "peak": peak, "unit": "GB/s",
                       "frac": achieved / peak, "traffic": NCU_TRAFFIC.get(args.config, {}).get(name),
                       "traffic_source": "profiles/r01_final_ncu_full_C4.md (ncu --set full, per launch)"
                       if args.config in NCU_TRAFFIC else None, "peak_source": peak_src,
                       "kernel_ms": dict(zip(KERNELS, kms)),
                       "kernel_share": {k: v / max(sum(kms), 1e-12) for k, v in zip(KERNELS, kms)},
                       "bytes_per_site": kb,
                       "step": {"floor_bytes_per_site": floor_bytes_per_site(cfg["model"]), "achieved": step_gbs,
                                "frac": step_gbs / peak}}
    if rank == 0:
        # north_star: "labelling-iteration counts" -- the union-find has no outer iteration, so what is
        # reported is one counted step: unions attempted / linked / retried in the global merge, find
        # hops there, and rounds of the root chase in the flip kernel
        g.set_counting(True)
        g.step(1)
        st = g.label_stats()
        g.set_counting(False)
        act = max(st["active_border_bonds"], 1)
        out["labelling"] = {"tile_face_bonds": st["border_bonds"], "active": st["active_border_bonds"],
                            "unions_linked": st["unions_linked"], "cas_retries": st["union_retries"],
                            "merge_hops_per_union": st["merge_find_hops"] / act, "merge_hops_max": st["merge_find_hops_max"],
                            "chase_rounds_per_thread": st["chase_hops"] / (n_sites / 16), "chase_rounds_max": st["chase_hops_max"],
                            "host_iterations": 0}
    if rank == 0 and not args.no_extras:
        # the paper's second row (Table 1): update + measurement of E and M every step,
        # through sw_run_series (per-step sums stay on the device)
        ns = max(3, min(args.steps, 20))
        g.run_series(ns)   # warm-up with the same length: the record buffer is sized once
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.run_series(ns)
        e1.record()
        torch.cuda.synchronize()
        ms_meas = e0.elapsed_time(e1) / ns
        out["with_measurement"] = {"ms_per_step": ms_meas, "value": n_sites / (ms_meas * 1e-3), "unit": UNIT,
                                   "what": "sw_run_series: every step followed by k_measure (E, and M for XY) and a snapshot"}
        out["e2e"] = measure_e2e(sw, torch, g, cfg, max(3, min(args.steps, 10)))
        if world == 1:
            spins, t = g.spins(), g.t
            out["cpu_baseline"] = oracle_baseline(cfg, spins, t)
            del spins
            others = {}
            for name_c, c in list(inputs.CONFIGS.items()) + list(inputs.EXTRA_CONFIGS.items()):
                if name_c == args.config:
                    continue
                g2, ms2, kms2, fl2 = time_config(sw, torch, c, args.seed, DEFAULT_BURN_IN[name_c], 3,
                                                 min(args.steps, 30), flush_buf)
                nn = c["L"] ** c["dim"]
                others[name_c] = {"workload": c["desc"], "ms_per_step": ms2, "site_updates_per_s": nn / (ms2 * 1e-3),
                                  "kernel_ms": dict(zip(KERNELS, kms2)),
                                  "step_floor_frac": floor_bytes_per_site(c["model"]) * nn / (ms2 * 1e-3) / 1e9 / peak}
                g2.close()
            out["other_configs"] = others
    g.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


def run_reference(args):
    """The oracle as the reference arm: rank 0 only, K timed steps after W warm-up steps, each step a
    bounded sample of the workload (the same model, dimension and temperature on a lattice small
    enough that the whole run ends within minutes)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    from oracle import sw_oracle as orc
    from paper_1403_7560_b200 import inputs
    cfg = dict({**inputs.CONFIGS, **inputs.EXTRA_CONFIGS}[args.config])
    budget = 150.0
    warm = max(args.warmup, 3)
    cands = [cfg["L"]] + ([256, 128, 64, 32] if cfg["dim"] == 3 else [2048, 1024, 512, 256, 128, 64])
    cands = [L for L in cands if L <= cfg["L"]]
    ns_guess = 200e-9
    L = next((L for L in cands if (args.steps + warm) * ns_guess * L ** cfg["dim"] <= budget), cands[-1])
    o = orc.Oracle(cfg["dim"], L, cfg["model"], cfg["q"], 1.0 / cfg["T"], args.seed)
    o.step(warm)
    t0 = time.perf_counter()
    o.step(args.steps)
    el = time.perf_counter() - t0
    n = o.N
    value = n * args.steps / el
    sample = (f"{args.steps} oracle steps (+{warm} warm-up) of {cfg['desc'].rsplit('L=', 1)[0]}L={L} at T={cfg['T']:.6f} "
              f"(workload {args.config} is L={cfg['L']}), 1 thread of {os.cpu_count()} host cores")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": warm, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {0: "int8", 1: "u8", 2: "f32", 3: "u16"}[cfg["model"]],
        "data": "synthetic", "config": {"workload": f"{args.config}: {cfg['desc']} (oracle sample L={L})", "sites": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)

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


# dram__bytes_read.sum + dram__bytes_write.sum per launch, from the `ncu --set full` captures summarised
# under profiles/ (config -> kernel -> bytes); lts__t_bytes for the L2-sized configs is in the same files.
NCU_TRAFFIC = {
    "C4": {"k_bond_label": 134.5e6 + 509.3e6, "k_merge": 348.1e6 + 68.4e6, "k_flip": 538.0e6 + 119.9e6},
    "C2": {"k_bond_label": 16.8e6 + 12.9e6, "k_merge": 49.0e6 + 0.2e6, "k_flip": 67.1e6 + 3.2e6},
    "C5": {"k_bond_label": 67.4e6 + 23.9e6, "k_merge": 38.6e6 + 0.1e6, "k_flip": 134.5e6 + 20.3e6},
    "X3": {"k_bond_label": 34.2e6 + 14.7e6, "k_merge": 38.7e6 + 0.1e6, "k_flip": 100.8e6 + 6.3e6},
    "C1": {"k_sw_small": 35.8e3 / 200},
}
NCU_TRAFFIC_SOURCE = {"C4": "profiles/r02_ncu_full_C4.md (ncu --set full, per launch)",
                      "C2": "profiles/r02_ncu_full_C2_C5_X3_C1.md (cold L2; L2 bytes in the same file)",
                      "C5": "profiles/r02_ncu_full_C2_C5_X3_C1.md (cold L2; L2 bytes in the same file)",
                      "X3": "profiles/r02_ncu_full_C2_C5_X3_C1.md (cold L2; L2 bytes in the same file)",
                      "C1": "profiles/r02_ncu_full_C2_C5_X3_C1.md (one launch of 200 steps, per step)"}


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


def _spread(xs):
    xs = sorted(xs)
    n = len(xs)
    mean = sum(xs) / n
    return {"min": xs[0], "median": xs[n // 2], "max": xs[-1], "mean": mean,
            "std": (sum((x - mean) ** 2 for x in xs) / max(n - 1, 1)) ** 0.5, "n": n}


def _events(torch, n):
    return [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]


def time_steps(torch, g, steps, flush_buf, needs_flush):
    """`steps` SW steps timed with CUDA events on the stream the library launches on (torch's current
    stream).  Returns (ms per step over the whole region, per-step spread or None)."""
    if g.info()["one_cta"]:
        # the lattice lives in the shared memory of one CTA: sw_step(steps) is ONE launch; the spread is over
        # five such launches
        per = []
        for a, b in _events(torch, 5):
            a.record()
            g.step(steps)
            b.record()
            torch.cuda.synchronize()
            per.append(a.elapsed_time(b) / steps)
        return per[len(per) // 2], _spread(per)
    if not needs_flush:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.step(steps)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        evs = _events(torch, steps)           # second pass: one event pair per step, for the spread
        for a, b in evs:
            a.record()
            g.step(1)
            b.record()
        torch.cuda.synchronize()
        return ms, _spread([a.elapsed_time(b) for a, b in evs])
    # working set comparable to L2: flush L2 (write a 512 MiB buffer) between timed steps
    evs = _events(torch, steps)
    for a, b in evs:
        flush_buf.add_(1)
        a.record()
        g.step(1)
        b.record()
    torch.cuda.synchronize()
    per = [a.elapsed_time(b) for a, b in evs]
    return sum(per) / steps, _spread(per)


def time_config(sw, torch, cfg, seed, burn_in, warmup, steps, flush_buf, first10=False, beta=None, start=None):
    """Thermalise, warm up, then time `steps` SW steps.  Returns (context, result dict)."""
    b = (1.0 / cfg["T"]) if beta is None else beta
    g = sw.SwendsenWang(cfg["dim"], cfg["L"], cfg["model"], cfg["q"], b, seed=seed)
    if start is not None:
        g.set_spins(start, 0)
    needs_flush = working_set_bytes(cfg) < 2 * L2_BYTES and not g.info()["one_cta"]
    res = {}
    if first10 and not g.info()["one_cta"]:
        # the seeded random start is the EASY case for the labelling (small clusters): steps 0-9
        g.step(0)
        torch.cuda.synchronize()
        evs = _events(torch, 10)
        for a, bb in evs:
            if needs_flush:
                flush_buf.add_(1)
            a.record()
            g.step(1)
            bb.record()
        torch.cuda.synchronize()
        res["first_10_steps_ms"] = _spread([a.elapsed_time(bb) for a, bb in evs])
        burn_in = max(burn_in - 10, 0)
    g.step(burn_in)
    g.step(warmup)
    torch.cuda.synchronize()
    ms, spread = time_steps(torch, g, steps, flush_buf, needs_flush)
    res["ms_per_step"] = ms
    res["ms_per_step_spread"] = spread
    # another pass over the same number of steps: per-kernel events (shares of the step)
    g.set_kernel_timing(True)
    if g.info()["one_cta"]:
        g.step(steps)
    else:
        for _ in range(steps):
            if needs_flush:
                flush_buf.add_(1)
            g.step(1)
    kms, ksteps = g.kernel_times()
    g.set_kernel_timing(False)
    res["kernel_ms"] = [x / max(ksteps, 1) for x in kms]
    res["flushed"] = needs_flush
    return g, res


def time_with_measurement(torch, g, ns):
    """The paper's second row (Table 1): update + measurement of E and M every step, through
    sw_run_series (per-step sums stay on the device)."""
    g.run_series(ns)   # warm-up with the same length: the record buffer is sized once
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.run_series(ns)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / ns


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
    return {"value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "h2d_bytes_per_step": nbytes + 8,
            "d2h_bytes_per_step": nbytes + g.info()["observables_copy_bytes"],
            "what": "per step: sw_set_spins (pinned host -> device, + the 8-byte step index), sw_step(1), "
                    "sw_observables (accumulator head -> host), sw_get_spins (device -> pinned host)"}


def oracle_baseline(cfg, spins, t, max_seconds=30.0):
    """The CPU oracle, as it stands, on a bounded sample of the same workload: whole-lattice steps
    from the GPU's thermalised configuration, one thread pinned to one core."""
    from oracle import sw_oracle as orc
    pinned = None
    try:
        allowed = sorted(os.sched_getaffinity(0))
        os.sched_setaffinity(0, {allowed[-1]})
        pinned = allowed
    except Exception:
        pass
    try:
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
    finally:
        if pinned is not None:
            os.sched_setaffinity(0, set(pinned))
    return {"value": n * done / el, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{done} whole-lattice oracle step(s) of {cfg['desc']} from the GPU's thermalised state, "
                      f"{el:.1f} s on 1 thread pinned to one of {os.cpu_count()} host cores"
                      + ("" if pinned is not None else " (pinning not available)"),
            "ns_per_site": 1e9 * el / (n * done)}


def max_over_ranks(ms, device):
    """Replicas only: the job's step time is the slowest rank's; the one
    collective of the multi-GPU path (not on the data path).  Works on NCCL (cuda) and gloo (cpu)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def kernel_names(info):
    return ("k_sw_small", "-", "-") if info["one_cta"] else KERNELS


def roofline_block(cfg, cfg_name, info, res, n_sites, peak, peak_src):
    """Roofline of the dominant kernel: algorithmic bytes / CUDA-event duration / measured copy peak."""
    kms = res["kernel_ms"]
    names = kernel_names(info)
    if info["one_cta"]:
        kb = {"k_sw_small": floor_bytes_per_site(cfg["model"])}
    else:
        kb = kernel_bytes_per_site(cfg["model"])
    dom = max(range(3), key=lambda k: kms[k])
    name = names[dom]
    achieved = kb[name] * n_sites / (kms[dom] * 1e-3) / 1e9 if kms[dom] > 0 else 0.0
    step_gbs = floor_bytes_per_site(cfg["model"]) * n_sites / (res["ms_per_step"] * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": name, "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak, "traffic": NCU_TRAFFIC.get(cfg_name, {}).get(name),
            "traffic_source": NCU_TRAFFIC_SOURCE.get(cfg_name), "peak_source": peak_src,
            "kernel_ms": {k: v for k, v in zip(names, kms) if k != "-"},
            "kernel_share": {k: v / max(sum(kms), 1e-12) for k, v in zip(names, kms) if k != "-"},
            "bytes_per_site": kb,
            "note": "one CTA, lattice resident in shared memory: latency-bound, the HBM roofline does not apply"
                    if info["one_cta"] else None,
            "step": {"floor_bytes_per_site": floor_bytes_per_site(cfg["model"]), "achieved": step_gbs,
                     "frac": step_gbs / peak}}


def run_micro(sw, peak):
    """The two bounds DESIGN.md section 6 quotes beside the HBM roofline, measured through sw_micro_bench."""
    n = 2 ** 27
    out = {}
    ms = sw.micro_bench(sw.MICRO_PHILOX_SITE, n, 0, 10)
    out["philox_per_site"] = {"ms": ms, "sites": n, "what": "one Philox4x32-10 call + 3 compares per site, 1 B/site written",
                              "sites_per_s": n / (ms * 1e-3)}
    ms = sw.micro_bench(sw.MICRO_PHILOX_GROUP, n, 0, 10)
    out["philox_per_group"] = {"ms": ms, "sites": n, "what": "transposed-digit decisions, 10 calls per 32 sites (reading 6), 12 B per 32 sites written",
                               "sites_per_s": n / (ms * 1e-3)}
    reads, words = 2 ** 26, 2 ** 27
    ms = sw.micro_bench(sw.MICRO_GATHER, reads, words, 10)
    out["random_gather"] = {"ms": ms, "reads": reads, "table_bytes": 4 * words, "reads_per_s": reads / (ms * 1e-3),
                            "what": "independent random 4-byte reads from a 512 MiB table (the access pattern of the root chase)"}
    return out


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
    allcfg = {**inputs.CONFIGS, **inputs.EXTRA_CONFIGS}
    cfg = allcfg[args.config]
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
        g, res = time_config(sw, torch, cfg, args.seed + rank, burn, warm, args.steps, flush_buf,
                             first10=(rank == 0 and not args.no_extras))
    ms = res["ms_per_step"]
    ms_all = max_over_ranks(ms, "cuda") if world > 1 else ms
    value = world * n_sites / (ms_all * 1e-3)
    info = g.info()
    launches = (5 + 1) if info["one_cta"] else 3 * args.steps

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_all, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {0: "int8", 1: "u8", 2: "f32", 3: "u16"}[cfg["model"]], "data": "synthetic",
        "config": {"workload": f"{args.config}: {cfg['desc']} periodic, T={cfg['T']:.6f}, Philox seed {args.seed}"
                               f" (+rank), seeded random start thermalised by {burn} untimed SW steps",
                   "sites": n_sites, "burn_in_steps": burn,
                   "l2": ("lattice resident in the shared memory of one CTA" if info["one_cta"] else
                          "L2 flushed (512 MiB write) between timed steps" if res["flushed"] else "inputs larger than L2 (no flush)"),
                   "tile": [info["tile_x"], info["tile_y"], info["tile_z"]], "rows_per_thread": info["rows_per_thread"],
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "gpu_launches": launches,
        "clocks": clk.summary(),
        "ms_per_step_spread": res["ms_per_step_spread"],
    }
    if "first_10_steps_ms" in res:
        out["first_10_steps_ms"] = res["first_10_steps_ms"]
    out["roofline"] = roofline_block(cfg, args.config, info, res, n_sites, peak, peak_src)
    if rank == 0 and not info["one_cta"]:
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
                            "chase_rounds_per_thread": st["chase_hops"] / (n_sites / info["flip_sites_per_thread"]),
                            "flip_sites_per_thread": info["flip_sites_per_thread"],
                            "chase_rounds_max": st["chase_hops_max"], "host_iterations": 0}
    if rank == 0 and not args.no_extras:
        ns = max(3, min(args.steps, 20))
        ms_meas = time_with_measurement(torch, g, ns)
        out["with_measurement"] = {"ms_per_step": ms_meas, "value": n_sites / (ms_meas * 1e-3), "unit": UNIT,
                                   "what": "sw_run_series: every step followed by the energy pass (E, and M for XY / clock) and a snapshot"}
        out["e2e"] = measure_e2e(sw, torch, g, cfg, max(3, min(args.steps, 10)))
        if world == 1:
            spins, t = g.spins(), g.t
            out["cpu_baseline"] = oracle_baseline(cfg, spins, t)
            del spins
            g.close()
            g = None
            # PAPER.md:187 "four independent runs": the same timing for seeds 1-4
            seeds = {}
            for sd in (1, 2, 3, 4):
                g2, r2 = time_config(sw, torch, cfg, sd, burn, 3, min(args.steps, 20), flush_buf)
                seeds[str(sd)] = r2["ms_per_step"]
                g2.close()
            out["seeds_ms_per_step"] = seeds
            others = {}
            for name_c, c in allcfg.items():
                if name_c == args.config:
                    continue
                nn = c["L"] ** c["dim"]
                g2, r2 = time_config(sw, torch, c, args.seed, DEFAULT_BURN_IN[name_c], 3, min(args.steps, 30), flush_buf, first10=True)
                i2 = g2.info()
                rb = roofline_block(c, name_c, i2, r2, nn, peak, peak_src)
                msm = time_with_measurement(torch, g2, max(3, min(args.steps, 20)))
                others[name_c] = {"workload": c["desc"], "ms_per_step": r2["ms_per_step"], "ms_per_step_spread": r2["ms_per_step_spread"],
                                  "first_10_steps_ms": r2.get("first_10_steps_ms"),
                                  "site_updates_per_s": nn / (r2["ms_per_step"] * 1e-3), "kernel_ms": rb["kernel_ms"],
                                  "with_measurement_ms_per_step": msm, "tile": [i2["tile_x"], i2["tile_y"], i2["tile_z"]],
                                  "one_cta": bool(i2["one_cta"]), "step_floor_frac": rb["step"]["frac"],
                                  "dominant_kernel": rb["kernel"], "dominant_kernel_frac": rb["frac"], "traffic": rb["traffic"]}
                g2.close()
            out["other_configs"] = others
            # SURVEY.md 8(d) stress inputs: the two extremes of the labelling cost at C2 / C4 size
            stress = {}
            for name_c in ("C2", "C4"):
                c = allcfg[name_c]
                nn = c["L"] ** c["dim"]
                for tag, beta, start in (("beta0", 0.0, None), ("cold_beta40", 40.0, inputs.aligned_spins(c["model"], nn))):
                    g2, r2 = time_config(sw, torch, c, args.seed, 3, 3, min(args.steps, 20), flush_buf, beta=beta, start=start)
                    stress[f"{name_c}_{tag}"] = {"ms_per_step": r2["ms_per_step"], "kernel_ms": dict(zip(KERNELS, r2["kernel_ms"])),
                                                 "what": "no bonds: N clusters" if beta == 0.0 else "every bond active: one cluster"}
                    g2.close()
            out["stress"] = stress
            out["micro"] = run_micro(sw, peak)
    if g is not None:
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

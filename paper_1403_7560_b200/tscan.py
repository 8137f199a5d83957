"""Temperature-scan driver: the paper's physics workflow in miniature.

The paper locates T_c from the crossing of the moment ratio U = <M^4> / <M^2>^2 (Eq. 6)
of several lattice sizes, with 10^4 discarded and 5x10^4 - 2x10^5 measured steps and four independent
runs per point.  This module runs that protocol on top of the C ABI
(sw_create / sw_run_series): one context per (L, T, seed), all Monte Carlo work in the CUDA kernels,
only the averaging here.  Production-scale statistics are out of scope.
"""
import numpy as np

from . import binding


def moment_ratio(m2, m4):
    """U = <M^4> / <M^2>^2 (Eq. 6)."""
    return float(np.mean(m4) / np.mean(m2) ** 2)


def _one_chain(dim, L, model, q, T, seed, n_discard, n_measure):
    """One (L, T, seed) chain on a context with its own CUDA stream (library-owned memory and stream)."""
    g = binding.SwendsenWang(dim, L, model, q, 1.0 / T, seed=seed, use_torch=False)
    g.step(n_discard)
    s = g.run_series(n_measure)
    g.close()
    N = L ** dim
    return moment_ratio(s["M2"], s["M4"]), float(np.mean(s["E"])) / N, float(np.mean(s["M2"])) / N ** 2


def scan(dim, model, sizes, temperatures, n_discard=1000, n_measure=10000, seeds=(1, 2, 3, 4), q=0, concurrent=16):
    """U(L, T), E/N and <M^2>/N^2 with errors from the spread over independent seeds.

    The paper's workflow is many temperatures x four independent runs: all (T, seed) chains
    of a size are independent, so up to `concurrent` of them are live at once, each on its own context and CUDA
    stream, driven by host threads (the C calls release the GIL).  Small lattices, which run in one CTA
    (sw_small.cuh) or are launch-bound, then share the GPU instead of queueing behind each other; the result
    does not depend on `concurrent` (same seeds, same series).

    Returns {L: {"T": array, "U": array, "U_err": array, "E": array, "E_err": array, "M2": array}}."""
    from concurrent.futures import ThreadPoolExecutor
    out = {}
    with ThreadPoolExecutor(max_workers=max(1, int(concurrent))) as pool:
        for L in sizes:
            jobs = {(T, seed): pool.submit(_one_chain, dim, L, model, q, T, seed, n_discard, n_measure)
                    for T in temperatures for seed in seeds}
            rows = []
            for T in temperatures:
                us, es, m2s = zip(*[jobs[(T, seed)].result() for seed in seeds])
                k = len(seeds)
                rows.append((T, np.mean(us), np.std(us, ddof=1) / np.sqrt(k) if k > 1 else 0.0,
                             np.mean(es), np.std(es, ddof=1) / np.sqrt(k) if k > 1 else 0.0, np.mean(m2s)))
            a = np.array(rows, dtype=np.float64)
            out[L] = {"T": a[:, 0], "U": a[:, 1], "U_err": a[:, 2], "E": a[:, 3], "E_err": a[:, 4], "M2": a[:, 5]}
    return out


def crossing(res, L1, L2):
    """Temperature where the U(T) curves of two sizes cross (linear interpolation of the difference
    between neighbouring scan points), and U there; None if they do not cross inside the scan."""
    T = res[L1]["T"]
    d = res[L1]["U"] - res[L2]["U"]
    for i in range(len(T) - 1):
        if d[i] == 0.0:
            return float(T[i]), float(res[L1]["U"][i])
        if d[i] * d[i + 1] < 0.0:
            w = d[i] / (d[i] - d[i + 1])
            return float(T[i] + w * (T[i + 1] - T[i])), float(res[L1]["U"][i] + w * (res[L1]["U"][i + 1] - res[L1]["U"][i]))
    return None


if __name__ == "__main__":
    import json
    import sys
    dim, model = 3, binding.ISING
    Ts = [4.40, 4.45, 4.49, 4.51, 4.53, 4.57, 4.62]
    r = scan(dim, model, [32, 64], Ts, n_discard=2000, n_measure=20000)
    for L, v in r.items():
        for T, U, e in zip(v["T"], v["U"], v["U_err"]):
            print(f"L={L:4d} T={T:.4f} U={U:.4f} +- {e:.4f}")
    print("crossing (T, U):", crossing(r, 32, 64), "  paper: T_c = 4.51151(1) (PAPER.md:195)")
    json.dump({str(L): {k: x.tolist() for k, x in v.items()} for L, v in r.items()}, sys.stdout if "--json" in sys.argv else open("/dev/null", "w"))

"""Small statistics helpers for the Monte Carlo tests (no method arithmetic here)."""
import numpy as np


def binned_mean_err(x, nbins=64):
    """Mean and its standard error from nbins non-overlapping bins (bin length >> tau_int)."""
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nbins) * nbins
    b = x[:n].reshape(nbins, -1).mean(axis=1)
    return float(b.mean()), float(b.std(ddof=1) / np.sqrt(nbins))


def pooled(series_list, nbins=64):
    """Pool independent runs: weighted by equal length; returns (mean, err)."""
    ms, es = zip(*[binned_mean_err(s, nbins) for s in series_list])
    k = len(ms)
    return float(np.mean(ms)), float(np.sqrt(np.sum(np.square(es))) / k)


def golden_rows(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append(line.split())
    return rows

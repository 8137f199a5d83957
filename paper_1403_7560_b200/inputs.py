"""Seeded synthetic input generators shared by the tests, bench.py and smoke() -- for BOTH the CUDA
path and the oracle.  This module holds none of the method's arithmetic (no bond probabilities, no
Philox, no labelling): only configurations to inject with set_spins, and the workload table of
BASELINE.json.  numpy only."""
import math

import numpy as np

ISING, POTTS, XY, CLOCK = 0, 1, 2, 3

# BASELINE.json configs: name -> (dim, L, model, q, T, steps)
CONFIGS = {
    "C1": dict(dim=2, L=64, model=ISING, q=0, T=2.269185, steps=1000, desc="2D Ising L=64"),
    "C2": dict(dim=2, L=4096, model=ISING, q=0, T=2.269185, steps=1000, desc="2D Ising L=4096"),
    "C3": dict(dim=2, L=4096, model=POTTS, q=3, T=1.0 / math.log(1.0 + math.sqrt(3.0)), steps=1000,
               desc="2D q=3 Potts L=4096"),
    "C4": dict(dim=3, L=512, model=ISING, q=0, T=4.5115, steps=500, desc="3D Ising L=512"),
    "C5": dict(dim=3, L=256, model=XY, q=0, T=2.2019, steps=500, desc="3D XY L=256"),
}


# The remaining two of the paper's six programs: timed by
# bench.py next to the five BASELINE configs, parity-tested at small sizes.
EXTRA_CONFIGS = {
    "X1": dict(dim=3, L=256, model=POTTS, q=3, T=1.8164, steps=500, desc="3D q=3 Potts L=256"),
    "X2": dict(dim=2, L=2048, model=XY, q=0, T=0.8929, steps=500, desc="2D XY L=2048"),
    # the model the paper's XY program and its Table 2 actually use: the 512-state clock model
    # (PAPER.md:159, 210), at the configuration of C5
    "X3": dict(dim=3, L=256, model=CLOCK, q=512, T=2.2019, steps=500, desc="3D 512-state clock L=256"),
}


def random_spins(model, N, q=0, seed=0):
    """Uniform random configuration (numpy PCG64, not the method's generator)."""
    rng = np.random.default_rng(seed)
    if model == ISING:
        return (2 * rng.integers(0, 2, size=N, dtype=np.int8) - 1).astype(np.int8)
    if model == POTTS:
        return rng.integers(0, q, size=N, dtype=np.uint8)
    if model == CLOCK:
        return rng.integers(0, q, size=N).astype(np.uint16)
    return (rng.random(N, dtype=np.float32) * np.float32(2.0 * math.pi)).astype(np.float32)


def aligned_spins(model, N, value=None):
    """Cold start: every spin equal (one cluster at large beta)."""
    if model == ISING:
        return np.full(N, 1 if value is None else value, dtype=np.int8)
    if model == POTTS:
        return np.full(N, 0 if value is None else value, dtype=np.uint8)
    if model == CLOCK:
        return np.full(N, 1 if value is None else value, dtype=np.uint16)
    return np.full(N, 0.5 if value is None else value, dtype=np.float32)


def striped_spins(model, dim, L, width, q=2):
    """Stripes of the given width along the last axis: long straight clusters that cross every tile."""
    N = L ** dim
    idx = np.arange(N, dtype=np.int64)
    c = (idx // L ** (dim - 1)) % L
    band = (c // width)
    if model == ISING:
        return (2 * (band % 2) - 1).astype(np.int8)
    if model == POTTS:
        return (band % q).astype(np.uint8)
    if model == CLOCK:
        return (band % q).astype(np.uint16)
    return ((band % 2) * np.float32(math.pi)).astype(np.float32)


def domain_spins(model, dim, L, block, q=2, seed=0):
    """Random value per block^dim domain: many mid-sized clusters with ragged tile crossings."""
    rng = np.random.default_rng(seed)
    nb = (L + block - 1) // block
    if model == ISING:
        vals = (2 * rng.integers(0, 2, size=nb ** dim) - 1).astype(np.int8)
    elif model == POTTS:
        vals = rng.integers(0, q, size=nb ** dim).astype(np.uint8)
    elif model == CLOCK:
        vals = rng.integers(0, q, size=nb ** dim).astype(np.uint16)
    else:
        vals = (rng.random(nb ** dim) * 2.0 * math.pi).astype(np.float32)
    idx = np.arange(L ** dim, dtype=np.int64)
    b = np.zeros_like(idx)
    for a in range(dim):
        b += (((idx // L ** a) % L) // block) * nb ** a
    return vals[b]

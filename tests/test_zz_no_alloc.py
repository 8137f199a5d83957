"""sw_cluster_stats_static (include/sw.h): the entry point that allocates no device memory.

Its scratch (one size counter per site) is a static device array inside libsw_b200.so, shared by all
calls, so the test makes TWO calls in a row on different labellings and sizes -- the second one on a
smaller lattice, whose counters the first call left dirty -- and compares both with the existing
path, sw_get_cluster_stats (scratch from cudaMalloc).  Integer sums: the results must be identical.
The file name keeps it last in pytest's collection order; it passes alone in a fresh process too
(nothing here depends on an earlier test having touched the library).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TC2 = 2.269185


def _static_stats(sw, torch, labels_host, stream=None):
    """Device tensors in, device tensor out: only the test allocates (through torch)."""
    lab32 = torch.from_numpy(np.ascontiguousarray(labels_host, dtype=np.uint32).view(np.int32).copy()).to("cuda")   # labels < 2^31
    out = torch.full((2,), -1, dtype=torch.int64, device="cuda")  # garbage on entry: the call must clear it
    st = stream if stream is not None else torch.cuda.current_stream()
    with torch.cuda.stream(st):
        sw.cluster_stats_static(lab32.data_ptr(), lab32.numel(), out.data_ptr(), st.cuda_stream)
    st.synchronize()
    return tuple(int(v) for v in out.cpu().tolist())


def test_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    import paper_1403_7560_b200 as sw

    # call 1: 3D Ising L = 64 (262144 sites) near T_c; call 2: 2D Potts q = 3, L = 256 (65536 sites), whose
    # counters overlap the ones call 1 used; call 3: the first lattice one step later, on another stream
    g1 = sw.SwendsenWang(3, 64, sw.ISING, 0, 1.0 / 4.5115, seed=11)
    g1.step(3)
    g2 = sw.SwendsenWang(2, 256, sw.POTTS, 3, 1.0 / 0.994973, seed=12)
    g2.step(5)
    want1, lab1 = g1.cluster_stats(), g1.labels()
    want2, lab2 = g2.cluster_stats(), g2.labels()
    got1 = _static_stats(sw, torch, lab1)
    got2 = _static_stats(sw, torch, lab2)
    assert got1 == want1, f"first call: static {got1} vs allocating path {want1}"
    assert got2 == want2, f"second call (dirty scratch): static {got2} vs allocating path {want2}"
    g1.step(1)
    want3 = g1.cluster_stats()
    got3 = _static_stats(sw, torch, g1.labels(), stream=torch.cuda.Stream())
    assert got3 == want3, f"third call (other stream): static {got3} vs allocating path {want3}"
    # and against the plain definition on the host
    sizes = np.bincount(lab2.astype(np.int64), minlength=lab2.size)
    assert got2 == (int(np.count_nonzero(sizes)), int((sizes.astype(np.int64) ** 2).sum()))


def test_static_scratch_largest_size_and_ragged_size():
    import torch
    import paper_1403_7560_b200 as sw

    n = sw.STATIC_MAX_SITES
    g = sw.SwendsenWang(2, 1024, sw.ISING, 0, 1.0 / TC2, seed=5)   # 2^20 sites = the limit
    assert g.N == n
    g.step(2)
    assert _static_stats(sw, torch, g.labels()) == g.cluster_stats()
    # a size that is no multiple of the block size, synthetic labels: clusters = runs of 7 sites
    m = 100003
    lab = (np.arange(m, dtype=np.uint32) // 7) * 7
    ncl = (m + 6) // 7
    s2 = (m // 7) * 49 + (m % 7) ** 2
    assert _static_stats(sw, torch, lab) == (ncl, s2)


def test_static_scratch_rejects_sizes_beyond_the_limit_and_null_pointers():
    import torch
    import paper_1403_7560_b200 as sw

    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    lab = torch.zeros(16, dtype=torch.int32, device="cuda")
    with pytest.raises(sw.SwError) as e:
        sw.cluster_stats_static(lab.data_ptr(), sw.STATIC_MAX_SITES + 1, out.data_ptr(), 0)
    assert "SW_STATIC_MAX_SITES" in str(e.value) and str(sw.STATIC_MAX_SITES) in str(e.value)
    with pytest.raises(sw.SwError):
        sw.cluster_stats_static(lab.data_ptr(), 0, out.data_ptr(), 0)
    with pytest.raises(sw.SwError):
        sw.cluster_stats_static(0, 16, out.data_ptr(), 0)
    with pytest.raises(sw.SwError):
        sw.cluster_stats_static(lab.data_ptr(), 16, 0, 0)
    torch.cuda.synchronize()
    assert out.tolist() == [0, 0]   # nothing was launched

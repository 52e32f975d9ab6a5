"""tlb_t1_events_static: the T1 search for callers that cannot allocate device memory.

Some users of the droplet analysis have no workspace to lend and may not call cudaMalloc: a tool that only compares two
Delaunay link lists and never builds a lattice, a monitor running next to a lattice that fills the GPU (an allocation
may fail there, and it stalls the device's streams even when it succeeds), a guest inside an application that owns all
device memory.  For them the library carries a fixed scratch array in its device image (include/tlb.h,
csrc/tlb_noalloc.cu).  The GPU test below runs that entry point twice in a row on the one shared array -- a large
problem first, a small different one second, so anything the first call left behind would show -- and compares every
output, bit for bit (integer work, the bar of tests/test_gpu_analysis.py), with tlb_t1_events, the handle-based path
(and the small one with the oracle as well).  The file sorts last on purpose: a failure here must not hide the other tests under `pytest -x`.
"""
import ctypes

import numpy as np
import pytest

import inputs
def _flipped_grid(cols, rows, n_flips, seed):
    """Link lists of a triangulated cols x rows grid (past) and of the same grid with n_flips diagonals flipped and the
    droplets renumbered (now); map[k] = past index of present droplet k, one droplet of a flipped square unmatched."""
    idx = lambda i, j: j * cols + i
    L = set()
    for j in range(rows):
        for i in range(cols):
            if i + 1 < cols: L.add((idx(i, j), idx(i + 1, j)))
            if j + 1 < rows: L.add((idx(i, j), idx(i, j + 1)))
            if i + 1 < cols and j + 1 < rows: L.add((idx(i, j), idx(i + 1, j + 1)))
    now = set(L)
    # squares two apart never share a side, so every flip is a clean T1
    squares = [(i, j) for j in range(0, rows - 1, 2) for i in range(0, cols - 1, 2)]
    order = np.argsort(inputs.uniform(seed, 11, np.arange(len(squares))))
    flips = [squares[k] for k in order[:n_flips]]
    for i, j in flips:
        now.remove((idx(i, j), idx(i + 1, j + 1)))
        now.add(tuple(sorted((idx(i + 1, j), idx(i, j + 1)))))
    n = cols * rows
    perm = np.argsort(inputs.uniform(seed, 12, np.arange(n))).astype(np.int32)
    inv = np.argsort(perm)
    now_r = np.array(sorted(tuple(sorted((inv[a], inv[b]))) for a, b in now), dtype=np.int32)
    past = np.array(sorted(L), dtype=np.int32)
    mp = perm.copy()
    i, j = flips[0]
    mp[inv[idx(i + 1, j + 1)]] = -1   # that flip must not be reported
    return past, now_r, mp, n, n_flips - 1


def test_static_limits_need_no_gpu():
    """Sizes beyond the fixed capacity are refused before any CUDA call, with a code and a message of their own."""
    from paper_2109_12565_b200 import binding
    binding.build()
    lib = binding.load_library()
    ne = ctypes.c_int32(7)
    rc = lib.tlb_t1_events_static(None, 0, None, 0, None, 0, binding.T1_STATIC_MAX_DROPLETS + 1, 0, ctypes.addressof(ne), None, None)
    assert rc == binding.TLB_ELIMIT and ne.value == 7
    assert b"tlb_t1_events_static" in lib.tlb_error_string(rc)
    assert lib.tlb_t1_events_static(None, 0, None, 0, None, 0, 4, 0, None, None, None) == binding.TLB_EINVAL
    assert lib.tlb_t1_events_static(None, 3, None, 0, None, 0, 4, 0, ctypes.addressof(ne), None, None) == binding.TLB_EINVAL


@pytest.mark.gpu
def test_static_t1_matches_handle_path_twice_in_a_row(oracle_mod):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2109_12565_b200 import binding
    binding.load_library()
    # only the existing path needs a handle: its tables live in the workspace, 32 ints per droplet <= nx ny
    t = binding.TLB(1024, 512)
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a), device=t.device)
    # the outputs are the caller's: allocated once, before the calls under test
    ne = torch.full((1,), -7, dtype=torch.int32, device=t.device)
    ev = torch.full((2048, 4), -7, dtype=torch.int32, device=t.device)
    for cols, rows, flips, seed in [(120, 90, 700, 1), (9, 7, 6, 2)]:   # 10800 droplets, then 63
        past, now, mp, n, expected = _flipped_grid(cols, rows, flips, seed)
        dp, dn, dm = dev(past), dev(now), dev(mp)
        ne.fill_(-7); ev.fill_(-7)
        binding.t1_events_static(dp, dn, n, ne, ev, dm)
        ref_ev, ref_ne = t.t1_events(dp, dn, n, dm, max_events=2048)
        k = int(ne.item())
        assert k == ref_ne == expected
        assert torch.equal(ev[:k], ref_ev)
        if n < 1000:   # the oracle's brute force takes minutes on the large case
            oev, one = oracle_mod.t1_events(past, now, mp)
            assert k == one and (ev[:k].cpu().numpy() == oev).all()
        assert (ev[k:] == -7).all()   # nothing written beyond the events found
    # a truncated output keeps the count and the sorted prefix; a frame against itself has no event
    binding.t1_events_static(dp, dn, n, ne, ev[:3], dm)
    assert int(ne.item()) == expected and torch.equal(ev[:3], ref_ev[:3])
    binding.t1_events_static(dp, dp, n, ne, ev)
    assert int(ne.item()) == 0
    # the largest size the array holds is accepted, one more is refused with the dedicated code
    binding.t1_events_static(dp, dn, binding.T1_STATIC_MAX_DROPLETS, ne, ev, dm)
    assert int(ne.item()) == expected and torch.equal(ev[:expected], ref_ev)
    with pytest.raises(binding.TLBError) as e:
        binding.t1_events_static(dp, dn, binding.T1_STATIC_MAX_DROPLETS + 1, ne, ev, dm)
    assert e.value.code == binding.TLB_ELIMIT

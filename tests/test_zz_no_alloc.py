"""crk_sfc_order_noalloc: the entry point for callers that cannot allocate device memory.

Some hosts of this library cannot let it call cudaMalloc: a simulation code that took the whole GPU for its own arena at
start-up has nothing left to give, and one that has other kernels in flight does not want the device-wide stall that
cudaMalloc / cudaFree bring.  For them the library keeps the working set of its radix sort in a fixed array inside its
own device image (CRK_NOALLOC_SCRATCH_BYTES, at most CRK_NOALLOC_MAX_N particles) and offers the curve order through it.

The checks: the permutation equals, bit for bit, what the allocating path (crk_build_cells + crk_get_perm on a fresh
context) gives -- integer work, so the bar is equality; this holds on two calls in a row with different inputs and sizes
(the array keeps the first call's contents: histograms, keys, the range flag) and again on the first input; a refused or
failed call leaves the next one intact.  The file name sorts after the other test files on purpose (pytest -x stops at
the first failure; this test must not hide the parity tests), and nothing here depends on what ran before it.
"""
import numpy as np
import pytest

import crk_workloads as wl

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _device_inputs(torch, ps):
    dev = torch.device("cuda:0")
    return [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).to(dev) for k in ("x", "y", "z", "h")]


def _perm_existing_path(torch, ps, t):
    from paper_2202_02840_b200 import Crk
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)      # fresh context: its key width comes from this input alone
    ctx.build_cells(*t)
    p = ctx.perm()
    torch.cuda.synchronize()
    out = p.cpu().numpy().copy()
    ctx.close()
    return out


def test_noalloc_order_equals_the_allocating_path_on_consecutive_calls():
    torch = _torch()
    from paper_2202_02840_b200 import crk_sfc_order_noalloc
    # three seeded sets: 8000 particles (3 full sort tiles of 2048 and a ragged one), a clustered set with a much smaller
    # h_min (more key bits, hence a different number of radix passes and the other ping-pong parity), and 64^3 = the maximum
    sets = [wl.tiny_uniform(n_side=20, seed=4101), wl.clustered_plummer(n_side=24, seed=4102), wl.tiny_uniform(n_side=64, seed=4103)]
    assert sets[2].n == 262144
    dev_in = [_device_inputs(torch, ps) for ps in sets]
    want = [_perm_existing_path(torch, ps, t) for ps, t in zip(sets, dev_in)]
    outs = [torch.full((ps.n,), -7, dtype=torch.int32, device="cuda:0") for ps in sets]     # the caller's buffers
    for rnd in range(2):                                  # the whole sequence twice: every call follows another one
        for k in (0, 1, 2, 0):
            outs[k].fill_(-7)
            crk_sfc_order_noalloc(*dev_in[k], sets[k].box, outs[k])
            got = outs[k].cpu().numpy()
            assert np.array_equal(got, want[k]), f"round {rnd} set {k}: {int((got != want[k]).sum())} of {got.size} entries differ"
            assert np.array_equal(np.sort(got), np.arange(sets[k].n, dtype=np.int32))     # and it is a permutation


def test_noalloc_refuses_what_does_not_fit_and_recovers_after_an_error():
    torch = _torch()
    from paper_2202_02840_b200 import crk_sfc_order_noalloc, CrkError, NOALLOC_MAX_N
    ps = wl.tiny_uniform(n_side=16, seed=4104)
    t = _device_inputs(torch, ps)
    want = _perm_existing_path(torch, ps, t)
    out = torch.empty(ps.n, dtype=torch.int32, device="cuda:0")
    # one particle too many: refused with a message that names the limit, before anything is launched
    big = [torch.full((NOALLOC_MAX_N + 1,), 0.25, device="cuda:0") for _ in range(4)]
    big_out = torch.full((NOALLOC_MAX_N + 1,), -7, dtype=torch.int32, device="cuda:0")
    with pytest.raises(CrkError) as ei:
        crk_sfc_order_noalloc(*big, 1.0, big_out)
    assert ei.value.code == -1 and "CRK_NOALLOC_MAX_N" in str(ei.value) and str(NOALLOC_MAX_N) in str(ei.value)
    assert int((big_out != -7).sum().item()) == 0
    # a position outside the box sets the range flag inside the shared array ...
    bad = [a.clone() for a in t]
    bad[0][5] = ps.box * 1.5
    with pytest.raises(CrkError) as ei:
        crk_sfc_order_noalloc(*bad, ps.box, out)
    assert ei.value.code == -2
    # ... and the next call clears it for itself
    crk_sfc_order_noalloc(*t, ps.box, out)
    assert np.array_equal(out.cpu().numpy(), want)
    # n = 0: nothing to do, no error
    e = torch.empty(0, device="cuda:0")
    crk_sfc_order_noalloc(e, e, e, e, 1.0, torch.empty(0, dtype=torch.int32, device="cuda:0"))

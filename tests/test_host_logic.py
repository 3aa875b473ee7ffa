"""CPU-side checks (no GPU): the C-ABI library exports every symbol include/crk.h declares, the binding lists the
same names, and the N > 1 bookkeeping of bench.py (independent seeded boxes per rank, MAX-over-ranks time, SUM-over-
ranks work) is right under a world_size-2 gloo group."""
import ctypes
import os
import re
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "crk.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(crk_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for need in ("crk_build_cells", "crk_volumes", "crk_rk_coefficients", "crk_hydro_derivs", "crk_step_derivs"):
        assert need in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2202_02840_b200 import build as crk_build
    from paper_2202_02840_b200 import binding
    lib_path = crk_build.build()
    assert os.path.exists(lib_path)
    lib = ctypes.CDLL(lib_path)          # loads without a GPU (no compute call is made)
    declared = _declared_functions()
    missing = [n for n in declared if not hasattr(lib, n)]
    assert not missing, missing
    assert sorted(binding.EXPORTED_SYMBOLS) == declared


def test_binding_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2202_02840_b200 import Crk
    with pytest.raises(Exception):
        Crk(box=1.0, gamma=5.0 / 3.0, n_h=2.4)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    import crk_workloads as wl
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ps = wl.make_config("tiny_uniform", 8, seed=bench.rank_seed("tiny_uniform", rank))
    ms, e2e = 10.0 + 5.0 * rank, 20.0 - 3.0 * rank
    pairs, npart = 1000.0 * (rank + 1), float(ps.n)
    out = bench.aggregate_over_ranks(ms, e2e, pairs, npart, world, "cpu")
    q.put((rank, out, float(ps.x[:16].sum())))
    dist.destroy_process_group()


def test_rank_bookkeeping_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, a0, s0), (_, a1, s1) = res
    assert a0 == a1 == (15.0, 20.0, 3000.0, 1024.0)      # MAX of times, SUM of work
    assert s0 != s1                                       # each rank generated its own box
    sys.path.insert(0, ROOT)
    import bench
    assert bench.rank_seed("cosmo", 0) == 1004            # rank 0 is the BASELINE seed

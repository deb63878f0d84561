"""CPU-side checks (no GPU): the C-ABI library loads and exports every symbol include/pdrt.h declares; the
control-point sharding of DESIGN.md §9 reproduces the single-process result with world_size 2 over gloo (the
per-rank compute is the float64 oracle here — test infrastructure — because the CUDA path needs a GPU)."""
import ctypes
import os
import re
import socket

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import paper_2512_18863_b200 as pkg
    from paper_2512_18863_b200 import build
    lib = build.build()
    header = open(os.path.join(ROOT, "include", "pdrt.h")).read()
    declared = sorted(set(re.findall(r"PDRT_API\s+[\w\s\*]+?\b(pdrt_\w+)\s*\(", header)))
    assert declared, "no PDRT_API declarations found"
    assert sorted(pkg.SYMBOLS) == declared, "binding.SYMBOLS and include/pdrt.h disagree"
    handle = ctypes.CDLL(lib)
    missing = [s for s in declared if not hasattr(handle, s)]
    assert not missing, f"libpdrt.so lacks {missing}"


def test_engine_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2512_18863_b200 import Engine, workloads as W
    wl = W.tiny(seed=1)
    with pytest.raises(Exception):
        Engine(wl.grid, wl.model, wl.density)


def test_shard_ranges_tile_the_arc():
    from paper_2512_18863_b200.shard import shard_range
    for n_cp in (1, 5, 178, 356):
        for world in (1, 2, 3, 4, 8):
            rs = [shard_range(n_cp, r, world) for r in range(world)]
            assert rs[0][0] == 0 and rs[-1][1] == n_cp
            assert all(a[1] == b[0] for a, b in zip(rs, rs[1:]))
            sizes = [hi - lo for lo, hi in rs]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import workloads as W
    from paper_2512_18863_b200.shard import gather_rows, reduce_dose, shard_range
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.tiny(seed=21, n_cp=5)
    orc = Oracle(wl.grid, wl.model, wl.density)
    lo, hi = shard_range(wl.n_cp, rank, world)
    part = torch.from_numpy(orc.dose(wl.leaves[lo:hi], wl.jaws[lo:hi], wl.gantry_deg[lo:hi], wl.mu[lo:hi]))
    dose = reduce_dose(part.clone())
    g = W.seeded_dose_gradient(wl, seed=21)
    dl, dj, dm = orc.dose_backward(wl.leaves[lo:hi], wl.jaws[lo:hi], wl.gantry_deg[lo:hi], wl.mu[lo:hi], g)
    dl, dj, dm = (gather_rows(torch.from_numpy(np.ascontiguousarray(a)), wl.n_cp) for a in (dl, dj, dm))
    if rank == 0:
        np.savez(out, dose=dose.numpy(), dl=dl.numpy(), dj=dj.numpy(), dm=dm.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_arc_equals_single_process_gloo(tmp_path):
    import torch.multiprocessing as mp
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import workloads as W
    out = str(tmp_path / "rank0.npz")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    wl = W.tiny(seed=21, n_cp=5)
    orc = Oracle(wl.grid, wl.model, wl.density)
    dose = orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    g = W.seeded_dose_gradient(wl, seed=21)
    dl, dj, dm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert np.allclose(got["dose"], dose, rtol=1e-12, atol=1e-14 * dose.max())
    assert np.array_equal(got["dl"], dl) and np.array_equal(got["dj"], dj) and np.array_equal(got["dm"], dm)

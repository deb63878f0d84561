"""CPU-side checks (no GPU): the C-ABI library loads and exports every symbol include/pdrt.h declares; the
control-point sharding of DESIGN.md §9 (the `ShardedDose` driver that bench.py --gpus N runs on every rank) reproduces
the single-process result with world_size 2 and 3 over gloo.  The per-rank engine is a stand-in with the Engine's call
signature that evaluates the float64 oracle — test infrastructure — because the CUDA path needs a GPU; the same driver
around the CUDA Engine is run with world_size 1 in tests/test_gpu_parity.py."""
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


class _OracleEngine:
    """Stand-in with the call signature of paper_2512_18863_b200.Engine (torch tensors in, `out=` filled)."""

    def __init__(self, wl):
        from oracle.oracle import Oracle
        self.orc = Oracle(wl.grid, wl.model, wl.density)
        self.dose_shape = self.orc.dose_shape

    def dose(self, leaves, jaws, gantry, mu, out):
        import torch
        out.copy_(torch.from_numpy(self.orc.dose(leaves.numpy(), jaws.numpy(), gantry.numpy(), mu.numpy())))
        return out

    def dose_backward(self, leaves, jaws, gantry, mu, g, out):
        import torch
        res = self.orc.dose_backward(leaves.numpy(), jaws.numpy(), gantry.numpy(), mu.numpy(), g.numpy())
        for o, r in zip(out, res):
            o.copy_(torch.from_numpy(np.ascontiguousarray(r)))
        return out


def _worker(rank, world, port, out, n_cp):
    import torch
    import torch.distributed as dist
    from paper_2512_18863_b200 import workloads as W
    from paper_2512_18863_b200.shard import ShardedDose
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.tiny(seed=21, n_cp=n_cp)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
    eng = _OracleEngine(wl)
    sh = ShardedDose(eng, t(wl.leaves), t(wl.jaws), t(wl.gantry_deg), t(wl.mu), eng.dose_shape, rank, world)
    sh.dose = sh.dose.double()                      # the stand-in is float64
    dose = sh.forward()
    sh.backward(torch.from_numpy(W.seeded_dose_gradient(wl, seed=21)))
    dl, dj, dm = sh.gather()
    if rank == 0:
        np.savez(out, dose=dose.numpy(), dl=dl.numpy(), dj=dj.numpy(), dm=dm.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,n_cp", [(2, 5), (3, 2)], ids=["world2", "world3_with_an_empty_rank"])
def test_sharded_arc_equals_single_process_gloo(tmp_path, world, n_cp):
    import torch.multiprocessing as mp
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import workloads as W
    out = str(tmp_path / "rank0.npz")
    mp.spawn(_worker, args=(world, _free_port(), out, n_cp), nprocs=world, join=True)
    got = np.load(out)
    wl = W.tiny(seed=21, n_cp=n_cp)
    orc = Oracle(wl.grid, wl.model, wl.density)
    dose = orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    g = W.seeded_dose_gradient(wl, seed=21)
    dl, dj, dm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert np.allclose(got["dose"], dose, rtol=1e-12, atol=1e-14 * dose.max())
    assert np.array_equal(got["dl"], dl) and np.array_equal(got["dj"], dj) and np.array_equal(got["dm"], dm)

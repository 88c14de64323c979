"""Multi-rank path on CPU (gloo, world_size 2): cell-range sharding reproduces the unsharded step
bit for bit (counter-based RNG keyed by GLOBAL cell id), and the diagnostics all-reduce
sums to the single-process value.  The per-shard step is run by the oracle here (no GPU on this box);
the GPU version of the same check is tests/test_gpu_parity.py::test_sharded_step_matches_unsharded."""
import os
import socket

import numpy as np
import pytest

import oracle
from paper_2602_21244_b200 import sharding, workloads as wl

torch = pytest.importorskip("torch")


def test_partition_covers_and_balances():
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=300_000)
    for world in (1, 2, 3, 8):
        b = sharding.partition_cells(pop.counts, world)
        assert b[0] == 0 and b[-1] == pop.n_cells and np.all(np.diff(b) >= 0)
        m = sharding.pairs_per_cell(pop.counts)
        per = np.array([m[b[r]:b[r + 1]].sum() for r in range(world)])
        assert per.sum() == m.sum()
        assert per.max() <= m.sum() / world + m.max()  # balanced to within one cell
    # degenerate inputs
    assert list(sharding.partition_cells(np.zeros(5, int), 2)) == [0, 0, 5] or sharding.partition_cells(np.zeros(5, int), 2)[-1] == 5
    assert list(sharding.partition_cells(np.array([], int), 3)) == [0, 0, 0, 0]
    assert np.array_equal(sharding.pairs_per_cell(np.array([0, 1, 2, 7]), 2), [0, 0, 1, 2])


def _prepare():
    pop = wl.mach10_cylinder(nx=24, ny=12, n_total=20_000, seed=7)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    tab = oracle.ChiTable(np.linspace(0.1, 2.5, 32 * 32, dtype=np.float32).reshape(32, 32), float(np.log(5.0)), float(np.log(6e4)))
    return pop, cs, v, tab


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    pop, cs, v, tab = _prepare()
    bounds = sharding.partition_cells(pop.counts, world)
    c0, lcs, lv = sharding.shard_sorted(cs, v, bounds, rank)
    prm = oracle.AbinitioParams(chi_mode=0, cell_base=c0)
    ref = oracle.collide_abinitio(lcs, *lv, prm, 11, 3, table=tab)
    e = float((ref.vx ** 2 + ref.vy ** 2 + ref.vz ** 2).sum())
    tot = sharding.allreduce_diagnostics([e, ref.vx.sum(), float((ref.pair_i >= 0).sum())])
    q.put((rank, int(bounds[rank]), int(cs[bounds[rank]]), ref.vx, ref.vy, ref.vz, tot))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_sharded_step_is_bit_identical():
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=120) for _ in procs], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    pop, cs, v, tab = _prepare()
    full = oracle.collide_abinitio(cs, *v, oracle.AbinitioParams(chi_mode=0), 11, 3, table=tab)
    for rank, c0, q0, vx, vy, vz, tot in got:
        np.testing.assert_array_equal(vx, full.vx[q0:q0 + len(vx)])
        np.testing.assert_array_equal(vy, full.vy[q0:q0 + len(vy)])
        np.testing.assert_array_equal(vz, full.vz[q0:q0 + len(vz)])
    e_full = float((full.vx ** 2 + full.vy ** 2 + full.vz ** 2).sum())
    np.testing.assert_allclose(got[0][6][0], e_full, rtol=1e-13)
    np.testing.assert_array_equal(got[0][6], got[1][6])
    assert got[0][6][2] == float((full.pair_i >= 0).sum())
    assert sum(len(g[3]) for g in got) == pop.n

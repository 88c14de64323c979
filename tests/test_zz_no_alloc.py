"""dsmc_bin_noalloc (-m gpu; collected last on purpose): the cell sort through the entry point that allocates nothing
(fixed file-scope scratch array, no context) against the existing path (Context.bin = dsmc_bin), bit for bit -- the
tolerance of every binning test here, the result being the unique stable sort -- on calls in a row that share the
scratch array, including a call that leaves an error status and stale records behind."""
import ctypes as C

import numpy as np
import pytest

from paper_2602_21244_b200 import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dsmc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2602_21244_b200 import dsmc as mod
    return mod


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _outs(n, n_cells):
    return (torch.full((n,), -7.0, dtype=torch.float32, device="cuda"), torch.full((n,), -7.0, dtype=torch.float32, device="cuda"),
            torch.full((n,), -7.0, dtype=torch.float32, device="cuda"), torch.full((n,), -7, dtype=torch.int32, device="cuda"),
            torch.full((n_cells + 1,), -7, dtype=torch.int32, device="cuda"))


def _reference(dsmc, pop):
    ctx = dsmc.Context(pop.n, pop.n_cells)
    ref = [t.clone() for t in ctx.bin(dev(pop.cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), pop.n_cells)]
    ctx.check()
    ctx.close()
    return ref


def test_bin_noalloc_equals_dsmc_bin_on_calls_in_a_row(dsmc):
    # two radix passes, several tiles, a ragged tail, empty cells; then ONE pass on a smaller input (stale records of
    # the first call stay in the array behind it); then the first again
    big = wl.mach10_cylinder(nx=60, ny=30, n_total=300_001)
    rng = np.random.default_rng(11)
    counts = rng.integers(0, 40, 300)
    counts[3], counts[4] = 0, 2048
    small = wl._populate("ragged", counts, np.full(300, 273.0), np.zeros(300), np.zeros(300), 5)
    pops = [big, small, big]
    refs = [_reference(dsmc, p) for p in pops[:2]]
    refs.append(refs[0])
    ins = [(dev(p.cell), dev(p.vx), dev(p.vy), dev(p.vz)) for p in pops]
    outs = [_outs(p.n, p.n_cells) for p in pops]
    status = [torch.full((1,), 99, dtype=torch.int32, device="cuda") for _ in pops]
    dsmc.noalloc_setup()
    for p, i, o in zip(pops[:2], ins, outs):  # warm-up: every kernel variant is loaded before memory is measured
        dsmc.bin_noalloc(*i, p.n_cells, o)
    torch.cuda.synchronize()
    for o in outs:
        for t in o:
            t.fill_(-7)
    free0 = torch.cuda.mem_get_info()[0]
    for p, i, o, st in zip(pops, ins, outs, status):  # back to back on one stream, no synchronisation in between
        dsmc.bin_noalloc(*i, p.n_cells, o, status=st)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free0 - free1 < (4 << 20), "the no-allocation entry point took %d bytes of device memory" % (free0 - free1)
    for k, (o, r, st) in enumerate(zip(outs, refs, status)):
        assert int(st.item()) == 0
        for name, got, want in zip(("vx_s", "vy_s", "vz_s", "perm", "cell_start"), o, r):
            assert torch.equal(got, want), "call %d: %s differs from dsmc_bin" % (k, name)


def test_bin_noalloc_status_is_per_call_and_limits_are_rejected(dsmc):
    pop = wl.mach10_cylinder(nx=40, ny=20, n_total=100_000)
    bad = pop.cell.copy()
    bad[12345] = pop.n_cells + 7
    bad[777] = -1
    i_bad = (dev(bad), dev(pop.vx), dev(pop.vy), dev(pop.vz))
    i_ok = (dev(pop.cell), dev(pop.vx), dev(pop.vy), dev(pop.vz))
    st = [torch.full((1,), 99, dtype=torch.int32, device="cuda") for _ in range(2)]
    o_bad, o_ok = _outs(pop.n, pop.n_cells), _outs(pop.n, pop.n_cells)
    dsmc.bin_noalloc(*i_bad, pop.n_cells, o_bad, status=st[0])
    dsmc.bin_noalloc(*i_ok, pop.n_cells, o_ok, status=st[1])  # the bad call's status and dropped records do not leak
    torch.cuda.synchronize()
    assert int(st[0].item()) == -2 and int(st[1].item()) == 0
    assert int(o_bad[4][-1].item()) == pop.n - 2  # the two bad ids were dropped, as dsmc_bin does
    for got, want in zip(o_ok, _reference(dsmc, pop)):
        assert torch.equal(got, want)
    # beyond the fixed scratch array: a clear error, nothing enqueued
    lib = dsmc._lib
    p = lambda t: C.c_void_p(t.data_ptr())
    args = [p(i_ok[0]), p(i_ok[1]), p(i_ok[2]), p(i_ok[3]), p(o_ok[0]), p(o_ok[1]), p(o_ok[2]), p(o_ok[3]), p(o_ok[4]), None]
    assert lib.dsmc_bin_noalloc(None, C.c_int64(dsmc.NOALLOC_MAX_PARTICLES + 1), C.c_int32(8), *args) == -7
    assert lib.dsmc_bin_noalloc(None, C.c_int64(100), C.c_int32(dsmc.NOALLOC_MAX_CELLS + 1), *args) == -7
    assert lib.dsmc_bin_noalloc(None, C.c_int64(-1), C.c_int32(8), *args) == -1
    assert "scratch" in dsmc.strerror(-7)
    # the largest size it accepts still sorts correctly (all of the scratch array in use)
    n, K = dsmc.NOALLOC_MAX_PARTICLES, dsmc.NOALLOC_MAX_CELLS
    rng = np.random.default_rng(2)
    cell = rng.integers(0, K, n).astype(np.int32)
    v = rng.standard_normal(n).astype(np.float32)
    o = _outs(n, K)
    dsmc.bin_noalloc(dev(cell), dev(v), dev(v), dev(v), K, o)
    torch.cuda.synchronize()
    perm = np.argsort(cell, kind="stable").astype(np.int32)
    assert np.array_equal(o[3].cpu().numpy(), perm)
    assert np.array_equal(o[4].cpu().numpy(), np.concatenate([[0], np.cumsum(np.bincount(cell, minlength=K))]).astype(np.int32))
    assert np.array_equal(o[0].cpu().numpy(), v[perm])

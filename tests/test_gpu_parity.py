"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI binding, against the CPU
oracle on the same seeded inputs.  Integer work (binning, pair indices, acceptance away from the
threshold) is bit-exact; FP32 velocities agree to 1e-5 per pair (Q21), conserved cell
moments to 1e-6; the BF16 tensor-core path to 2e-2 per pair."""
import math

import numpy as np
import pytest

import os

import oracle
from conftest import _OBSERVED
from paper_2602_21244_b200 import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KB = 1.380649e-23
M = wl.MASS_AR


@pytest.fixture(scope="module")
def dsmc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2602_21244_b200 import dsmc as mod
    return mod


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _note(what, value, tol):
    """worst observed error of the running test, kept beside its tolerance (conftest: gpurun_out/parity_observed.txt)"""
    name = os.environ.get("PYTEST_CURRENT_TEST", "?").split("::")[-1].split(" ")[0]
    _OBSERVED("%s %s" % (name, what), value, tol)


def binned(dsmc, ctx, pop):
    out = ctx.bin(dev(pop.cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), pop.n_cells)
    ctx.check()
    return out


# --------------------------------------------------------------------------------------- a1
@pytest.mark.parametrize("case", ["tiny", "couette", "mach10_small", "ragged", "empty", "three_pass", "one_pass"])
def test_bin_bit_exact(dsmc, case):
    if case == "tiny":
        pop = wl.tiny_box()
    elif case == "couette":
        pop = wl.couette(n_cells=50, per_cell=1000)
    elif case == "mach10_small":
        pop = wl.mach10_cylinder(nx=80, ny=40, n_total=400_000)
    elif case == "ragged":
        rng = np.random.default_rng(7)
        counts = rng.integers(0, 40, 3001)
        counts[17] = 2048
        counts[18] = 0
        counts[19] = 1
        pop = wl._populate("ragged", counts, np.full(3001, 300.0), np.zeros(3001), np.zeros(3001), 7)
    elif case == "three_pass":   # 300 000 cells need 19 bits: three radix passes
        rng = np.random.default_rng(11)
        counts = rng.integers(0, 4, 300_000)
        pop = wl._populate("three_pass", counts, np.full(300_000, 300.0), np.zeros(300_000), np.zeros(300_000), 11)
    elif case == "one_pass":     # 300 cells: a single pass that is both first and last
        rng = np.random.default_rng(12)
        counts = rng.integers(0, 900, 300)
        pop = wl._populate("one_pass", counts, np.full(300, 300.0), np.zeros(300), np.zeros(300), 12)
    else:
        pop = wl._populate("empty", np.zeros(5, np.int64), np.full(5, 300.0), np.zeros(5), np.zeros(5), 1)
    ctx = dsmc.Context(max(pop.n, 1), pop.n_cells)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    rc, perm_o, cs_o = oracle.bin_particles(pop.cell, pop.n_cells)
    assert rc == 0
    np.testing.assert_array_equal(cs.cpu().numpy(), cs_o)
    np.testing.assert_array_equal(perm.cpu().numpy(), perm_o)
    np.testing.assert_array_equal(vx_s.cpu().numpy(), pop.vx[perm_o])
    np.testing.assert_array_equal(vy_s.cpu().numpy(), pop.vy[perm_o])
    np.testing.assert_array_equal(vz_s.cpu().numpy(), pop.vz[perm_o])
    ctx.close()


def test_bin_reports_bad_cell_index_and_large_cells(dsmc):
    pop = wl.tiny_box(n_cells=4, per_cell=10)
    cell = pop.cell.copy()
    cell[3] = 4
    ctx = dsmc.Context(pop.n, 4)
    ctx.bin(dev(cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), 4)
    assert ctx.sync_status() == dsmc.ERR_BAD_CELL_INDEX
    assert ctx.sync_status() == 0  # sticky status is cleared by the read
    cell[3] = -1
    ctx.bin(dev(cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), 4)
    assert ctx.sync_status() == dsmc.ERR_BAD_CELL_INDEX
    # a cell above DSMC_MAX_CELL_PARTICLES sorts fine but is refused by the SMEM-resident fused step
    big = wl._populate("big", np.array([5000, 5]), np.full(2, 300.0), np.zeros(2), np.zeros(2), 1)
    ctx2 = dsmc.Context(big.n, 2)
    vx_s, vy_s, vz_s, perm, cs = ctx2.bin(dev(big.cell), dev(big.vx), dev(big.vy), dev(big.vz), 2)
    assert ctx2.sync_status() == 0
    rc, perm_o, cs_o = oracle.bin_particles(big.cell, 2)
    np.testing.assert_array_equal(perm.cpu().numpy(), perm_o)
    tab = _lj_table(16, 16)
    ctx2.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    ctx2.collide_abinitio(cs, vx_s, vy_s, vz_s, dsmc.AbinitioParams(), 0, 0)
    assert ctx2.sync_status() == dsmc.ERR_CELL_TOO_LARGE


def test_bin_bad_cell_index_multi_pass_is_memory_safe(dsmc):
    """Bad ids with K > 512 (two radix passes): the first pass drops them, so the later pass reads a stale tail of the
    ping-pong buffers.  Run after another context of the same process has used and freed its workspace (stale, valid-
    looking data in recycled memory): the call must report the error and leave the CUDA context healthy."""
    rng = np.random.default_rng(21)
    warm = wl.mach10_cylinder(nx=80, ny=40, n_total=300_000)
    ctx0 = dsmc.Context(warm.n, warm.n_cells)
    binned(dsmc, ctx0, warm)
    ctx0.close()
    K = 3000
    counts = rng.integers(50, 150, K)
    pop = wl._populate("bad_multi", counts, np.full(K, 300.0), np.zeros(K), np.zeros(K), 21)
    cell = pop.cell.copy()
    bad = rng.choice(pop.n, 5000, replace=False)
    cell[bad[:2500]] = K + rng.integers(0, 1 << 20, 2500)
    cell[bad[2500:]] = -1 - rng.integers(0, 1000, 2500)
    ctx = dsmc.Context(pop.n, K)
    ctx.bin(dev(cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), K)
    assert ctx.sync_status() == dsmc.ERR_BAD_CELL_INDEX
    # the context still works: a clean input sorts bit-exactly afterwards
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    rc, perm_o, cs_o = oracle.bin_particles(pop.cell, K)
    np.testing.assert_array_equal(cs.cpu().numpy(), cs_o)
    np.testing.assert_array_equal(perm.cpu().numpy(), perm_o)
    ctx.close()


# --------------------------------------------------------------------------------------- a2 / a8
def test_cell_moments_and_standalone_match(dsmc):
    pop = wl.mach10_cylinder(nx=40, ny=20, n_total=150_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    mom = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
    cs_h = cs.cpu().numpy()
    v = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
    mom_o = oracle.cell_moments(cs_h, *v)
    np.testing.assert_allclose(mom, mom_o, rtol=1e-12, atol=1e-6)
    # stand-alone correction towards the moments of a different population
    other = wl.mach10_cylinder(seed=9, nx=40, ny=20, n_total=150_000)
    rc, perm2, _ = oracle.bin_particles(other.cell, other.n_cells)
    tgt = oracle.cell_moments(cs_h, *[a[perm2].astype(np.float64) for a in (other.vx, other.vy, other.vz)])
    for flags in (dsmc.F_MOMENT_MATCH, dsmc.F_MOMENT_MATCH | dsmc.F_MATCH_ENERGY_ONLY):
        x, y, z = vx_s.clone(), vy_s.clone(), vz_s.clone()
        ctx.moment_match(cs, x, y, z, dev(tgt), flags)
        ctx.check()
        ref = oracle.moment_match(cs_h, *v, tgt, flags)
        N = np.diff(cs_h)
        scale = np.repeat(np.sqrt(np.maximum(tgt[:, 3], 1) / np.maximum(N, 1)), N)
        for got, want in zip((x, y, z), ref):
            assert np.abs(got.cpu().numpy() - want).max() <= 2e-6 * scale.max()
            assert (np.abs(got.cpu().numpy() - want) / scale).max() <= 2e-6
        got_m = ctx.cell_moments(cs, x, y, z).cpu().numpy()
        ok = N >= 2
        np.testing.assert_allclose(got_m[ok, 3], tgt[ok, 3], rtol=1e-6)
        if not flags & dsmc.F_MATCH_ENERGY_ONLY:
            assert (np.abs(got_m[ok, :3] - tgt[ok, :3]).max(axis=1) / (N[ok] * np.sqrt(tgt[ok, 3] / N[ok]))).max() < 1e-6


# --------------------------------------------------------------------------------------- fused steps
def _setup_vhs(dsmc, pop, H, seed_w, n_in=8, act=None):
    ctx = dsmc.Context(pop.n, pop.n_cells)
    Ws, bs = wl.random_mlp(seed_w, [n_in, H, H, 3] if isinstance(H, int) else [n_in, H[0], H[1], 3])
    act = dsmc.ACT_TANH if act is None else act
    ctx.set_mlp(0, Ws, bs, act)
    return ctx, oracle.Mlp(Ws, bs, act)


def _compare_step(dsmc, ctx, cs, v_in, v_out, dump, ref, tol_pair, tol_moment, gate=None, slope=None):
    """Shared checks: bit-exact pairing, per-pair g' error (Q21), cell moments."""
    cs_h = cs.cpu().numpy()
    pi, pj, acc = dump.pair_i.cpu().numpy(), dump.pair_j.cpu().numpy(), dump.accepted.cpu().numpy()
    np.testing.assert_array_equal(pi, ref.pair_i)
    np.testing.assert_array_equal(pj, ref.pair_j)
    np.testing.assert_array_equal(acc, ref.accepted)
    idx = np.flatnonzero(ref.pair_i >= 0)
    k = np.searchsorted(cs_h, idx, side="right") - 1
    g = np.stack([a[cs_h[k] + pi[idx]] - a[cs_h[k] + pj[idx]] for a in v_in], axis=1)
    gn = np.linalg.norm(g, axis=1)
    err = np.linalg.norm(dump.gprime.cpu().numpy()[idx].astype(np.float64) - ref.gprime[idx], axis=1) / np.maximum(gn, 1e-30)
    allow = np.full(len(idx), tol_pair)
    if slope is not None:
        allow = allow + slope[idx]
    sel = np.ones(len(idx), bool) if gate is None else gate[idx]
    assert sel.mean() > 0.97, "too many pairs excluded from the gate"
    bad = err[sel] > allow[sel]
    if slope is None:
        _note("pair |dg'|/g", err[sel].max() if sel.any() else 0.0, tol_pair)
    else:
        _note("pair |dg'|/g over its allowance", (err[sel] / allow[sel]).max() if sel.any() else 0.0, 1.0)
    assert not bad.any(), "per-pair error: max %.3e (allowed %.1e), %d bad" % (err[sel].max(), tol_pair, bad.sum())
    return err


def _velocity_and_moment_checks(ctx, cs, v_in, out, ref, tol_pair, tol_moment):
    """Final velocities against the oracle's, in units of the cell's thermal scale s = sqrt(E/N).  The tolerance follows
    from the per-pair one (DESIGN "Tolerances"): v' = cm +- g'/2, so a pair whose g' is off by tol_pair * g moves its two
    particles by tol_pair * g / 2; the matching then rescales by alpha = 1 + O(tol_moment) and shifts by O(tol_moment) s,
    and fp32 storage adds 6e-8 |v|.  Hence tol_v = tol_pair * max(g / s) / 2 + 2e-6, g / s from the oracle's pairs."""
    cs_h = cs.cpu().numpy()
    N = np.diff(cs_h)
    pre = oracle.cell_moments(cs_h, *v_in)
    got = ctx.cell_moments(cs, *out).cpu().numpy()
    ok = N >= 2
    _note("cell energy", np.abs(got[ok, 3] / pre[ok, 3] - 1).max(), tol_moment)
    _note("cell momentum", (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max(), tol_moment)
    assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < tol_moment
    assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < tol_moment
    cell_scale = np.sqrt(np.maximum(pre[:, 3], 1e-30) / np.maximum(N, 1))
    scale = np.repeat(cell_scale, N)
    idx = np.flatnonzero(ref.pair_i >= 0)
    k = np.searchsorted(cs_h, idx, side="right") - 1
    g = np.sqrt(sum((a[cs_h[k] + ref.pair_i[idx]] - a[cs_h[k] + ref.pair_j[idx]]) ** 2 for a in v_in))
    tol_v = 0.5 * tol_pair * (g / cell_scale[k]).max() + 2e-6
    assert tol_v < 5e-5  # never looser than the fixed figure this replaced
    for a, want in zip(out, (ref.vx, ref.vy, ref.vz)):
        d = np.abs(a.cpu().numpy().astype(np.float64) - want) / scale
        _note("velocity / thermal scale", d.max(), tol_v)
        assert d.max() < tol_v, "velocity mismatch %.3e (allowed %.3e)" % (d.max(), tol_v)


@pytest.mark.parametrize("case", ["cfg1_tiny", "cfg2_couette_small", "cfg3_cavity_small", "ragged"])
def test_collide_vhs_nn_fp32(dsmc, case):
    if case == "cfg1_tiny":
        pop, H, ppc, sw = wl.tiny_box(), 64, 50, 0
    elif case == "cfg2_couette_small":
        pop, H, ppc, sw = wl.couette(n_cells=12, per_cell=1000), 128, 500, 1
    elif case == "cfg3_cavity_small":
        pop, H, ppc, sw = wl.cavity(nx=20, ny=20), 128, 50, 2
    else:
        rng = np.random.default_rng(3)
        counts = rng.integers(0, 30, 400)
        counts[5], counts[6], counts[7], counts[8] = 0, 1, 2, 3
        counts[100] = 2048
        pop, H, ppc, sw = wl._populate("ragged", counts, np.full(400, 273.0), np.zeros(400), np.zeros(400), 3), 64, -1, 0
    ctx, net = _setup_vhs(dsmc, pop, H, sw)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    prm = dsmc.VhsParams(sigma_v=wl.SIGMA_V, pairs_per_cell=ppc)
    oprm = oracle.VhsParams(sigma_v=float(np.float32(wl.SIGMA_V)), pairs_per_cell=ppc)
    for step in range(3):  # per-step re-sync (Q20): the oracle is fed the GPU's input state
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        dump = dsmc.PairDump(pop.n, "cuda")
        ctx.collide_vhs_nn(cs, vx_s, vy_s, vz_s, prm, seed=sw, step=step, dump=dump)
        ctx.check()
        ref = oracle.collide_vhs_nn(cs_h, *v_in, net, oprm, sw, step)
        hn = ref.aux
        med = np.median(hn[ref.pair_i >= 0])
        err = _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, gate=hn >= 0.25 * med)
        _velocity_and_moment_checks(ctx, cs, v_in, (vx_s, vy_s, vz_s), ref, 1e-5, 1e-6)
    ctx.close()


def test_collide_vhs_nn_variants(dsmc):
    """paper's 6-input ReLU form (Q1), shell off, matching off / energy-only, acceptance."""
    pop = wl.couette(seed=5, n_cells=16, per_cell=300)
    for n_in, act, flags in ((6, 1, dsmc.F_NOISE | dsmc.F_ENERGY_SHELL),
                             (8, 2, dsmc.F_NOISE | dsmc.F_MOMENT_MATCH),
                             (8, 0, dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | dsmc.F_MATCH_ENERGY_ONLY),
                             (8, 0, dsmc.F_NOISE | dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | dsmc.F_ACCEPT)):
        ctx, net = _setup_vhs(dsmc, pop, 32, 4, n_in=n_in, act=act)
        vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
        cs_h = cs.cpu().numpy()
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        prm = dsmc.VhsParams(sigma_v=wl.SIGMA_V, flags=flags)
        oprm = oracle.VhsParams(sigma_v=float(np.float32(wl.SIGMA_V)), flags=flags)
        cap = None
        if flags & dsmc.F_ACCEPT:
            cap = np.full(pop.n_cells, oracle.vhs_sigma_g(6 * wl.SIGMA_V, oprm), np.float32)
        dump = dsmc.PairDump(pop.n, "cuda")
        ctx.collide_vhs_nn(cs, vx_s, vy_s, vz_s, prm, seed=11, step=2, sigma_cr_max=dev(cap) if cap is not None else None, dump=dump)
        ctx.check()
        ref = oracle.collide_vhs_nn(cs_h, *v_in, net, oprm, 11, 2, sigma_cr_max=cap)
        if flags & dsmc.F_ACCEPT:  # Q22: decisions within 1e-5 of the threshold may differ
            diff = dump.accepted.cpu().numpy() != ref.accepted
            assert diff.sum() <= 2
            assert 0.3 < ref.accepted[ref.pair_i >= 0].mean() < 0.9
            if diff.any():
                continue
        hn = ref.aux
        sel = ref.pair_i >= 0
        gate = (hn >= 0.25 * np.median(hn[sel & (ref.accepted == 1)])) | (ref.accepted == 0)
        if not flags & dsmc.F_ENERGY_SHELL:
            gate = np.ones_like(gate)
        _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, gate=gate)
        for a, want in zip((vx_s, vy_s, vz_s), (ref.vx, ref.vy, ref.vz)):
            assert np.abs(a.cpu().numpy() - want).max() < 2e-4 * 400
        ctx.close()


def _lj_table(nE=128, nB=128):
    return oracle.build_chi_table(oracle.lj_argon(), nE, nB, n_panels=2)


def _table_slope(tab, lnE, bt):
    """max-min of the four nodes surrounding each query (Q25 slope-aware tolerance)."""
    nE, nB = tab.chi.shape
    tE = np.clip((lnE - tab.lnE_min) / (tab.lnE_max - tab.lnE_min) * (nE - 1), 0, nE - 1)
    tB = np.clip(bt * (nB - 1), 0, nB - 1)
    iE = np.minimum(tE.astype(int), nE - 2)
    iB = np.minimum(tB.astype(int), nB - 2)
    c = np.stack([tab.chi[iE, iB], tab.chi[iE, iB + 1], tab.chi[iE + 1, iB], tab.chi[iE + 1, iB + 1]])
    return c.max(axis=0) - c.min(axis=0)


def _q25_bound(tab, cs_h, v_in, ref, seed, step):
    """Q25 on every pair, from the oracle's side alone: |chi_gpu - chi_oracle| <= 1e-5 max(|chi|, 1) + 2e-4 (max - min of
    the four table nodes around the query) + 1e-6.  Returns (indices of the pair slots, bound, pair speed g)."""
    idx = np.flatnonzero(ref.pair_i >= 0)
    k = np.searchsorted(cs_h, idx, side="right") - 1
    g2 = sum((a[cs_h[k] + ref.pair_i[idx]] - a[cs_h[k] + ref.pair_j[idx]]) ** 2 for a in v_in)
    bt = np.sqrt(oracle.pair_uniforms_batch(seed, step, k, idx - cs_h[k])[:, 1])
    sl = _table_slope(tab, np.log(np.maximum(M * g2 / (4 * KB), 1e-300)), bt)
    return idx, 1e-5 * np.maximum(np.abs(ref.aux[idx]), 1) + 2e-4 * sl + 1e-6, np.sqrt(g2)


@pytest.mark.parametrize("mode", ["table", "mlp"])
def test_collide_abinitio_fp32(dsmc, mode):
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=300_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    tab = _lj_table()
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    cm = 0 if mode == "table" else 1
    prm = dsmc.AbinitioParams(chi_mode=cm)
    oprm = oracle.AbinitioParams(chi_mode=cm, lnE_min=float(np.float32(prm.lnE_min)), lnE_max=float(np.float32(prm.lnE_max)))
    otab = oracle.ChiTable(tab.chi, float(np.float32(tab.lnE_min)), float(np.float32(tab.lnE_max)))
    for step in range(2):
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        dump = dsmc.PairDump(pop.n, "cuda")
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, seed=4, step=step, dump=dump)
        ctx.check()
        ref = oracle.collide_abinitio(cs_h, *v_in, oprm, 4, step, net=net, table=otab)
        slope = None
        chi_g = dump.aux.cpu().numpy().astype(np.float64)
        sel = ref.pair_i >= 0
        if mode == "table":  # Q25: fp32 table coordinates move the query by ~1e-4 grid cells
            idx = np.flatnonzero(sel)
            dchi = np.abs(chi_g - ref.aux)
            assert (dchi[idx] > 1e-5 * np.maximum(np.abs(ref.aux[idx]), 1)).mean() < 0.01
            assert dchi[idx].max() < 2e-3
            # the slope-aware bound of Q25 on EVERY pair, from the oracle's inputs alone (table nodes around the
            # query, pair uniforms): it bounds chi, and with it the angle by which g' may differ
            idx, bound, _ = _q25_bound(tab, cs_h, v_in, ref, 4, step)
            assert np.all(dchi[idx] <= bound), "chi outside the Q25 bound: %d pairs" % (dchi[idx] > bound).sum()
            slope = np.zeros_like(dchi)
            slope[idx] = bound  # a lookup difference rotates g' by exactly that angle
        else:
            rel = np.abs(chi_g[sel] - ref.aux[sel]) / np.maximum(np.abs(ref.aux[sel]), 1)
            _note("chi / max(|chi|,1), per pair", rel.max(), 1e-5)
            assert rel.max() <= 1e-5
        _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, slope=slope)
        N = np.diff(cs_h)
        pre = oracle.cell_moments(cs_h, *v_in)
        got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
        ok = N >= 2
        assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
        assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
        # untouched cells (N<2) are bit-identical
        lone = np.flatnonzero(N == 1)
        for k1 in lone[:50]:
            assert vx_s[cs_h[k1]].item() == np.float32(v_in[0][cs_h[k1]])
    ctx.close()


@pytest.mark.parametrize("mode", ["table", "mlp_tc", "mlp_tc_one_kernel"])
def test_abinitio_acceptance_and_partial_pairs(dsmc, mode):
    """NTC acceptance and a pair count below N / 2 (uniform request, then a per-cell array with zeros): pairs and
    decisions against the oracle, per-pair g' (table: FP32; tensor cores: chi within Q26), moments of every cell, and
    cells in which nothing was accepted stay bit-identical.  The tensor-core forms see gaps in their pair arrays here."""
    pop = wl.tiny_box(seed=12, n_cells=30, per_cell=501, T=500.0)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    tab = _lj_table(64, 64)
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    gmax = np.full(pop.n_cells, 6 * math.sqrt(2 * KB * 500.0 / M), np.float32)
    cm = 0 if mode == "table" else 1
    flags = dsmc.F_MOMENT_MATCH | dsmc.F_ACCEPT
    gflags = flags | (dsmc.F_BF16_TC if cm else 0) | (dsmc.F_TC_ONE_KERNEL if mode == "mlp_tc_one_kernel" else 0)
    otab = oracle.ChiTable(tab.chi, float(np.float32(tab.lnE_min)), float(np.float32(tab.lnE_max)))
    counts = np.full(pop.n_cells, 100, np.int32)
    counts[[2, 3, 17]] = 0
    counts[5] = 1
    counts[9] = 250
    for step, (ppc, pc) in enumerate(((100, None), (-1, counts))):
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        before = [t.clone() for t in (vx_s, vy_s, vz_s)]
        dump = dsmc.PairDump(pop.n, "cuda")
        prm = dsmc.AbinitioParams(chi_mode=cm, flags=gflags, pairs_per_cell=ppc)
        oprm = oracle.AbinitioParams(chi_mode=cm, flags=flags, pairs_per_cell=ppc, lnE_min=float(np.float32(prm.lnE_min)),
                                     lnE_max=float(np.float32(prm.lnE_max)))
        if pc is not None:
            prm.pairs_count = dev(pc)
            oprm.pairs_count = pc
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, 8, step, cr_max=dev(gmax), dump=dump)
        ctx.check()
        ref = oracle.collide_abinitio(cs_h, *v_in, oprm, 8, step, table=otab, net=net, cr_max=gmax)
        np.testing.assert_array_equal(dump.pair_i.cpu().numpy(), ref.pair_i)
        np.testing.assert_array_equal(dump.pair_j.cpu().numpy(), ref.pair_j)
        assert (ref.pair_i >= 0).sum() == (3000 if pc is None else int(counts.sum()))
        diff = dump.accepted.cpu().numpy() != ref.accepted
        assert diff.sum() <= 1  # Q22
        if diff.any():
            continue
        chi_g = dump.aux.cpu().numpy().astype(np.float64)
        sel = (ref.pair_i >= 0) & (ref.accepted == 1)
        if cm:
            assert (np.abs(chi_g[sel] - ref.aux[sel]) / (1 + np.abs(ref.aux[sel]))).max() <= 2e-2
            slope = 1.01 * np.abs(chi_g - ref.aux)
        else:
            idx, bound, _ = _q25_bound(tab, cs_h, v_in, ref, 8, step)
            acc_idx = ref.accepted[idx] == 1
            assert np.all(np.abs(chi_g - ref.aux)[idx][acc_idx] <= bound[acc_idx])
            slope = np.zeros_like(chi_g)
            slope[idx] = bound
        _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, slope=slope)
        N = np.diff(cs_h)
        pre = oracle.cell_moments(cs_h, *v_in)
        got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
        assert np.abs(got[:, 3] / pre[:, 3] - 1).max() < 1e-6
        assert (np.linalg.norm(got[:, :3] - pre[:, :3], axis=1) / (N * np.sqrt(pre[:, 3] / N))).max() < 1e-6
        if pc is not None:  # cells that were asked for no pairs are untouched
            for k in (2, 3, 17):
                for a, b in zip((vx_s, vy_s, vz_s), before):
                    assert torch.equal(a[cs_h[k]:cs_h[k + 1]], b[cs_h[k]:cs_h[k + 1]])
    ctx.close()


# --------------------------------------------------------------------------------------- a10
@pytest.mark.parametrize("mode", ["table", "mlp"])
def test_chi_batch(dsmc, mode):
    n = 200_003
    E, b = wl.abinitio_pair_batch(seed=3, n=n)
    E[:4] = [1.0, 1e6, 5.0, 6e4]  # clamped edges
    ctx = dsmc.Context(n, 1)
    tab = _lj_table()
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    got = ctx.chi_batch(dev(E), dev(b), 0 if mode == "table" else 1, 1e-9).cpu().numpy().astype(np.float64)
    ctx.check()
    lo, hi = float(np.float32(tab.lnE_min)), float(np.float32(tab.lnE_max))
    if mode == "table":
        want = oracle.chi_batch(E, b, 0, 1e-9, table=oracle.ChiTable(tab.chi, lo, hi))
        sl = _table_slope(tab, np.log(E.astype(np.float64)), b.astype(np.float64) / 1e-9)
        assert np.all(np.abs(got - want) <= 1e-5 * np.maximum(np.abs(want), 1) + 2e-4 * sl + 1e-6)
    else:
        want = oracle.chi_batch(E, b, 1, 1e-9, net=oracle.Mlp(Ws, bs, oracle.ACT_SILU), lnE_min=lo, lnE_max=hi)
        _note("chi / max(|chi|,1), per pair", (np.abs(got - want) / np.maximum(np.abs(want), 1)).max(), 1e-5)
        assert np.all(np.abs(got - want) <= 1e-5 * np.maximum(np.abs(want), 1))


def test_empty_inputs_and_unconfigured_operators(dsmc):
    ctx = dsmc.Context(16, 4)
    z = torch.zeros(0, dtype=torch.float32, device="cuda")
    cs = torch.zeros(5, dtype=torch.int32, device="cuda")
    ctx.collide_abinitio(cs, z, z, z, dsmc.AbinitioParams(), 0, 0)  # n == 0: OK, nothing launched
    v = torch.ones(8, dtype=torch.float32, device="cuda")
    cs = dev(np.array([0, 2, 4, 6, 8], np.int32))
    with pytest.raises(dsmc.DsmcError) as e:
        ctx.collide_abinitio(cs, v, v.clone(), v.clone(), dsmc.AbinitioParams(), 0, 0)
    assert e.value.status == dsmc.ERR_NOT_CONFIGURED
    with pytest.raises(dsmc.DsmcError):
        ctx.collide_vhs_nn(cs, v, v.clone(), v.clone(), dsmc.VhsParams(), 0, 0)
    Ws, bs = wl.random_mlp(0, [8, 200, 200, 3])
    ctx.set_mlp(0, Ws, bs, dsmc.ACT_TANH)
    with pytest.raises(dsmc.DsmcError) as e:  # the BF16 TC paths take hidden widths up to 128 only
        ctx.collide_vhs_nn(cs, v, v.clone(), v.clone(), dsmc.VhsParams(flags=dsmc.F_BF16_TC), 0, 0)
    assert e.value.status == dsmc.ERR_UNSUPPORTED_SHAPE


# --------------------------------------------------------------------------- BF16 tcgen05 paths
def _quantiles(x):
    return "median %.2e, 99%% %.2e, 99.9%% %.2e, max %.2e" % tuple(np.quantile(x, [0.5, 0.99, 0.999, 1.0]))


_DEEP = {"paper5": [2, 128, 96, 64, 48, 32, 1],   # five hidden layers, decreasing width, SiLU
         "deep4": [2, 64, 64, 48, 16, 1], "three": [2, 128, 128, 100, 1], "narrow": [2, 40, 24, 1]}


@pytest.mark.parametrize("H,act", [(128, "silu"), (64, "silu"), (128, "tanh"), (64, "relu"), ("paper5", "silu"),
                                   ("deep4", "tanh"), ("three", "relu"), ("narrow", "silu")])
def test_chi_batch_bf16_tc(dsmc, H, act):
    """a10 on the tensor cores; tolerance Q26: abs(dchi) <= 2e-2 (1 + abs(chi)).  Shapes: the BASELINE 2-H-H-1 and
    networks with up to five hidden layers of unequal widths <= 128 (zero-padded on the device), among them the
    paper's chi-MLP shape."""
    n = 300_017  # 2343 full tiles + a ragged tail of 113 pairs
    E, b = wl.abinitio_pair_batch(seed=3, n=n)
    E[:4] = [1.0, 1e6, 5.0, 6e4]
    a_g = {"silu": dsmc.ACT_SILU, "tanh": dsmc.ACT_TANH, "relu": dsmc.ACT_RELU}[act]
    a_o = {"silu": oracle.ACT_SILU, "tanh": oracle.ACT_TANH, "relu": oracle.ACT_RELU}[act]
    ctx = dsmc.Context(n, 1)
    Ws, bs = wl.random_mlp(3, _DEEP[H] if isinstance(H, str) else [2, H, H, 1])
    ctx.set_mlp(1, Ws, bs, a_g)
    got = ctx.chi_batch(dev(E), dev(b), 1, 1e-9, flags=dsmc.F_BF16_TC).cpu().numpy().astype(np.float64)
    ctx.check()
    lo, hi = float(np.float32(np.log(5.0))), float(np.float32(np.log(6.0e4)))
    want = oracle.chi_batch(E, b, 1, 1e-9, net=oracle.Mlp(Ws, bs, a_o), lnE_min=lo, lnE_max=hi)
    rel = np.abs(got - want) / (1 + np.abs(want))
    print("chi bf16 H=%s %s: %s" % (H, act, _quantiles(rel)))
    assert rel.max() <= 2e-2
    ctx.close()


@pytest.mark.parametrize("one_kernel", [False, True])
def test_collide_abinitio_bf16_tc(dsmc, one_kernel):
    """chi-MLP on the tensor cores, both forms: the default three passes (pairing + inputs | chi batch | rotation +
    matching) and, with F_TC_ONE_KERNEL, the single kernel of cell teams + MLP server."""
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=300_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    prm = dsmc.AbinitioParams(chi_mode=1, flags=dsmc.F_MOMENT_MATCH | dsmc.F_BF16_TC | (dsmc.F_TC_ONE_KERNEL if one_kernel else 0))
    oprm = oracle.AbinitioParams(chi_mode=1, lnE_min=float(np.float32(prm.lnE_min)), lnE_max=float(np.float32(prm.lnE_max)))
    for step in range(2):
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        dump = dsmc.PairDump(pop.n, "cuda")
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, seed=4, step=step, dump=dump)
        ctx.check()
        ref = oracle.collide_abinitio(cs_h, *v_in, oprm, 4, step, net=net)
        sel = ref.pair_i >= 0
        chi_g = dump.aux.cpu().numpy().astype(np.float64)
        rel = np.abs(chi_g[sel] - ref.aux[sel]) / (1 + np.abs(ref.aux[sel]))
        print("abinitio bf16 chi: %s" % _quantiles(rel))
        assert rel.max() <= 2e-2  # Q26
        # a chi difference rotates g' by exactly that angle: allow it on top of the fp32 rotation error
        # (the chi error of EVERY pair has just passed the Q26 bound, which is computed from the oracle's chi alone)
        err = _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, slope=1.01 * np.abs(chi_g - ref.aux))
        assert np.all(err <= 2e-2 * (1 + np.abs(ref.aux[sel])) + 1e-5)  # per pair, from the oracle's side alone
        N = np.diff(cs_h)
        pre = oracle.cell_moments(cs_h, *v_in)
        got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
        ok = N >= 2
        assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
        assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
    ctx.close()


def test_collide_abinitio_bf16_tc_paper_shape(dsmc):
    """The fused chi-MLP step on the tensor cores with the paper's chi-MLP shape (five hidden layers of decreasing width,
    SiLU): pairs bit-exact, chi within Q26 on every pair, moments; with-replacement selection too; the
    one-kernel form has no image for this shape and says so."""
    pop = wl.mach10_cylinder(nx=40, ny=20, n_total=120_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    Ws, bs = wl.random_mlp(7, _DEEP["paper5"])
    Ws = [w * np.float32(2.5) for w in Ws]  # (a random-init deep network is nearly constant: raise the gain of every layer)
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    for step, extra in enumerate((0, dsmc.F_PAIR_REPLACE)):
        prm = dsmc.AbinitioParams(chi_mode=1, flags=dsmc.F_MOMENT_MATCH | dsmc.F_BF16_TC | extra)
        oprm = oracle.AbinitioParams(chi_mode=1, flags=oracle.F_MOMENT_MATCH | (oracle.F_PAIR_REPLACE if extra else 0),
                                     lnE_min=float(np.float32(prm.lnE_min)), lnE_max=float(np.float32(prm.lnE_max)))
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        dump = dsmc.PairDump(pop.n, "cuda")
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, seed=5, step=step, dump=dump)
        ctx.check()
        ref = oracle.collide_abinitio(cs_h, *v_in, oprm, 5, step, net=net)
        sel = ref.pair_i >= 0
        chi_g = dump.aux.cpu().numpy().astype(np.float64)
        assert (np.abs(chi_g[sel] - ref.aux[sel]) / (1 + np.abs(ref.aux[sel]))).max() <= 2e-2  # Q26
        assert np.ptp(ref.aux[sel]) > 0.05
        _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, slope=1.01 * np.abs(chi_g - ref.aux))
        N = np.diff(cs_h)
        pre = oracle.cell_moments(cs_h, *v_in)
        got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
        ok = N >= 2
        assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
        assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
    with pytest.raises(dsmc.DsmcError) as e:
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, dsmc.AbinitioParams(chi_mode=1, flags=dsmc.F_BF16_TC | dsmc.F_TC_ONE_KERNEL), seed=5, step=9)
    assert e.value.status == dsmc.ERR_UNSUPPORTED_SHAPE
    ctx.close()


@pytest.mark.parametrize("one_kernel", [False, True])
def test_collide_abinitio_bf16_tc_few_cells_and_ragged(dsmc, one_kernel):
    """Both tensor-core forms on contexts whose radix sort needs a single pass (<= 512 cells: the split form's pair
    arrays must exist all the same) and on ragged cells (empty, 1, 2, 3, odd, 2048 particles)."""
    rng = np.random.default_rng(3)
    counts = rng.integers(0, 30, 200)
    counts[5], counts[6], counts[7], counts[8], counts[50], counts[120] = 0, 1, 2, 3, 2048, 777
    pop = wl._populate("ragged", counts, np.full(200, 273.0), np.zeros(200), np.zeros(200), 3)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    prm = dsmc.AbinitioParams(chi_mode=1, flags=dsmc.F_MOMENT_MATCH | dsmc.F_BF16_TC | (dsmc.F_TC_ONE_KERNEL if one_kernel else 0))
    oprm = oracle.AbinitioParams(chi_mode=1, lnE_min=float(np.float32(prm.lnE_min)), lnE_max=float(np.float32(prm.lnE_max)))
    v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
    dump = dsmc.PairDump(pop.n, "cuda")
    ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, seed=6, step=1, dump=dump)
    ctx.check()
    ref = oracle.collide_abinitio(cs_h, *v_in, oprm, 6, 1, net=net)
    sel = ref.pair_i >= 0
    chi_g = dump.aux.cpu().numpy().astype(np.float64)
    assert (np.abs(chi_g[sel] - ref.aux[sel]) / (1 + np.abs(ref.aux[sel]))).max() <= 2e-2  # Q26
    _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, slope=1.01 * np.abs(chi_g - ref.aux))
    N = np.diff(cs_h)
    pre = oracle.cell_moments(cs_h, *v_in)
    got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
    ok = N >= 2
    assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
    assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
    ctx.close()


@pytest.mark.parametrize("one_kernel", [False, True])
@pytest.mark.parametrize("case", ["cfg1_tiny", "cfg3_cavity_small", "ragged6", "narrow"])
def test_collide_vhs_nn_bf16_tc(dsmc, case, one_kernel):
    """BF16 tensor-core VHS-NN, both forms (default: three passes around a persistent split-precision batch kernel;
    F_TC_ONE_KERNEL: the chunk kernel with its own engine): bit-exact pairing, 2e-2 per pair on the gated set (Q21),
    1e-6 on moments; with NTC acceptance in the last step."""
    n_in = 8
    if case == "cfg1_tiny":
        pop, H, ppc, sw = wl.tiny_box(), 64, 50, 0
    elif case == "cfg3_cavity_small":
        pop, H, ppc, sw = wl.cavity(nx=20, ny=20), 128, 50, 2
    elif case == "narrow":  # unequal hidden widths below 64 / 128: zero-padded on the device
        pop, H, ppc, sw = wl.cavity(nx=12, ny=12), (100, 72), 50, 4
    else:
        rng = np.random.default_rng(3)
        counts = rng.integers(0, 30, 400)
        counts[5], counts[6], counts[7], counts[8] = 0, 1, 2, 3
        counts[100] = 2048
        pop, H, ppc, sw, n_in = wl._populate("ragged", counts, np.full(400, 273.0), np.zeros(400), np.zeros(400), 3), 64, -1, 0, 6
    ctx, net = _setup_vhs(dsmc, pop, H, sw, n_in=n_in)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    flags = dsmc.F_NOISE | dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | dsmc.F_BF16_TC | (dsmc.F_TC_ONE_KERNEL if one_kernel else 0)
    prm = dsmc.VhsParams(sigma_v=wl.SIGMA_V, pairs_per_cell=ppc, flags=flags)
    oprm = oracle.VhsParams(sigma_v=float(np.float32(wl.SIGMA_V)), pairs_per_cell=ppc)
    for step in range(3):
        v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
        dump = dsmc.PairDump(pop.n, "cuda")
        cap = None
        if step == 2:  # NTC acceptance on top
            prm = dsmc.VhsParams(sigma_v=wl.SIGMA_V, pairs_per_cell=ppc, flags=flags | dsmc.F_ACCEPT)
            oprm = oracle.VhsParams(sigma_v=float(np.float32(wl.SIGMA_V)), pairs_per_cell=ppc,
                                    flags=oracle.F_NOISE | oracle.F_ENERGY_SHELL | oracle.F_MOMENT_MATCH | oracle.F_ACCEPT)
            cap = np.full(pop.n_cells, oracle.vhs_sigma_g(6 * wl.SIGMA_V, oprm), np.float32)
        ctx.collide_vhs_nn(cs, vx_s, vy_s, vz_s, prm, seed=sw, step=step, sigma_cr_max=dev(cap) if cap is not None else None, dump=dump)
        ctx.check()
        ref = oracle.collide_vhs_nn(cs_h, *v_in, net, oprm, sw, step, sigma_cr_max=cap)
        if cap is not None:
            diff = dump.accepted.cpu().numpy() != ref.accepted
            assert diff.sum() <= 2  # Q22
            assert 0.2 < ref.accepted[ref.pair_i >= 0].mean() < 0.95
            if diff.any():
                continue
        hn = ref.aux
        med = np.median(hn[ref.pair_i >= 0])
        gate = (hn >= 0.25 * med) | (ref.accepted == 0)
        err = _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 2e-2, 1e-6, gate=gate)
        print("vhs bf16 %s one_kernel=%s: all pairs %s; excluded %.2f%%" % (case, one_kernel, _quantiles(err), 100 * (1 - gate[ref.pair_i >= 0].mean())))
        N = np.diff(cs_h)
        pre = oracle.cell_moments(cs_h, *v_in)
        got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
        ok = N >= 2
        assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
        assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
    ctx.close()


# --------------------------------------------------------------------------------------- (e) sharding
@pytest.mark.parametrize("tc", [False, True, "one_kernel"])
def test_sharded_step_matches_unsharded(dsmc, tc):
    """Two cell-range shards run one after the other on this GPU (independent launches, no rank waits on
    another) give bit-identical velocities to the unsharded step: RNG is keyed by the GLOBAL cell id."""
    from paper_2602_21244_b200 import sharding
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=300_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    tab = _lj_table(64, 64)
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    flags = dsmc.F_MOMENT_MATCH | (dsmc.F_BF16_TC if tc else 0) | (dsmc.F_TC_ONE_KERNEL if tc == "one_kernel" else 0)
    full = [t.clone() for t in (vx_s, vy_s, vz_s)]
    ctx.collide_abinitio(cs, *full, dsmc.AbinitioParams(chi_mode=1 if tc else 0, flags=flags), seed=9, step=2)
    ctx.check()
    bounds = sharding.partition_cells(np.diff(cs_h), 2)
    host = [t.cpu().numpy() for t in (vx_s, vy_s, vz_s)]
    for rank in range(2):
        c0, lcs, lv = sharding.shard_sorted(cs_h, host, bounds, rank)
        lt = [dev(a) for a in lv]
        ctx.collide_abinitio(dev(lcs), *lt, dsmc.AbinitioParams(chi_mode=1 if tc else 0, flags=flags, cell_base=c0), seed=9, step=2)
        ctx.check()
        q0 = int(cs_h[bounds[rank]])
        for a, b in zip(lt, full):
            assert torch.equal(a, b[q0:q0 + a.shape[0]])
    ctx.close()


# --------------------------------------------------------------------------------------- (f3) exact chi
def test_chi_exact_batch_golden_and_oracle(dsmc):
    """dsmc_chi_exact_batch (deflection-integral quadrature on the GPU, FP64 inside, fp32 in / out) against
    (a) the LJ worked values of tests/golden (SURVEY pin P8) and (b) the oracle's quadrature on a grid of
    (E*, b*) away from the orbiting band (Q23).  fp32 inputs limit the agreement to ~1e-6."""
    import os
    eps_k, sig = 119.8, 3.405e-10
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "lj_chi_worked_values.txt"))
            if l.strip() and not l.startswith("#")]
    Es = np.array([float(r[0]) for r in rows]); bs = np.array([float(r[1]) for r in rows]); want = np.array([float(r[2]) for r in rows])
    ctx = dsmc.Context(1 << 16, 1)
    E32, b32 = (Es * eps_k).astype(np.float32), (bs * sig).astype(np.float32)
    got = ctx.chi_exact_batch(dev(E32), dev(b32), eps_k, sig).cpu().numpy().astype(np.float64)
    ctx.check()
    assert np.abs(got - want).max() < 5e-6, np.abs(got - want).max()
    # grid against the oracle, evaluated at the fp32-rounded inputs; E* >= 1 keeps clear of the orbiting band
    rng = np.random.default_rng(5)
    n = 4000
    Er = np.exp(rng.uniform(np.log(1.0), np.log(500.0), n)); br = rng.uniform(0.0, 2.9, n)
    E32, b32 = (Er * eps_k).astype(np.float32), (br * sig).astype(np.float32)
    b32[:5] = 0.0
    got = ctx.chi_exact_batch(dev(E32), dev(b32), eps_k, sig).cpu().numpy().astype(np.float64)
    pot = oracle.lj_argon()
    ref = np.array([oracle.chi_exact(pot, float(e) * KB, float(b)) for e, b in zip(E32, b32)])
    d = np.abs(got - ref)
    print("chi exact vs oracle: median %.2e, 99.9%% %.2e, max %.2e" % (np.median(d), np.quantile(d, 0.999), d.max()))
    assert np.all(got[:5] == np.float32(np.pi))
    assert np.quantile(d, 0.999) < 5e-6 and d.max() < 1e-3  # a handful of points sit next to the orbiting curve
    absd = ctx.chi_exact_batch(dev(E32), dev(b32), eps_k, sig, flags=dsmc.F_CHI_ABS).cpu().numpy()
    assert np.array_equal(absd, np.abs(got.astype(np.float32)))
    ctx.close()


def test_build_chi_table_on_device(dsmc):
    """(f2) the chi table generated on the GPU by the quadrature kernel against the oracle's table builder, node by
    node outside the orbiting band (Q23), and lookups through the installed table against the oracle's bilinear."""
    nE = nB = 128
    lo, hi = float(np.float32(np.log(5.0))), float(np.float32(np.log(6.0e4)))
    ctx = dsmc.Context(1 << 16, 1)
    got = ctx.build_chi_table_lj(nE, nB, lo, hi, 1e-9, want_nodes=True).cpu().numpy().astype(np.float64)
    ctx.check()
    tab = oracle.build_chi_table(oracle.lj_argon(), nE, nB, lnE_min=lo, lnE_max=hi, b_max=1e-9, n_panels=2)
    want = tab.chi.astype(np.float64)
    d = np.abs(got - want)
    # orbiting band: rows with E* < 0.8 near the orbiting impact parameter are ill-conditioned (chi -> infinity);
    # compare where the table is smooth (neighbouring nodes within 0.5 rad)
    smooth = np.ones_like(d, bool)
    smooth[:, 1:] &= np.abs(np.diff(want, axis=1)) < 0.5
    smooth[:, :-1] &= np.abs(np.diff(want, axis=1)) < 0.5
    print("device-built chi table: max diff on smooth nodes %.2e (%.1f%% of nodes), elsewhere median %.2e"
          % (d[smooth].max(), 100 * smooth.mean(), np.median(d[~smooth]) if (~smooth).any() else 0.0))
    assert smooth.mean() > 0.97
    assert d[smooth].max() < 5e-6
    assert got[:, 0].min() == np.float32(np.pi) and got[:, 0].max() == np.float32(np.pi)  # b = 0: head-on
    # the installed table serves lookups
    E, b = wl.abinitio_pair_batch(seed=9, n=50_000)
    chi = ctx.chi_batch(dev(E), dev(b), 0, 1e-9).cpu().numpy().astype(np.float64)
    ref = oracle.chi_batch(E, b, 0, 1e-9, table=oracle.ChiTable(got.astype(np.float32), lo, hi))
    sl = _table_slope(oracle.ChiTable(got.astype(np.float32), lo, hi), np.log(E.astype(np.float64)), b.astype(np.float64) / 1e-9)
    assert np.all(np.abs(chi - ref) <= 1e-5 * np.maximum(np.abs(ref), 1) + 2e-4 * sl + 1e-6)
    ctx.close()


@pytest.mark.parametrize("tc", [False, True])
def test_build_chi_table_from_the_chi_mlp(dsmc, tc):
    """(f2 as the paper states it) the chi table generated on the device by the slot-1 chi-MLP against the
    oracle's orc_build_chi_table_mlp on EVERY node (FP32: 1e-5 max(chi, 1); tensor cores: Q26), lookups through the
    installed table, the cap (Q23) on a network that exceeds it, and the error paths."""
    nE, nB = 96, 80
    lo, hi = float(np.float32(np.log(5.0))), float(np.float32(np.log(6.0e4)))
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx = dsmc.Context(1 << 16, 1)
    with pytest.raises(RuntimeError):
        ctx.build_chi_table_mlp(nE, nB, lo, hi)  # no slot-1 network yet
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    got = ctx.build_chi_table_mlp(nE, nB, lo, hi, flags=dsmc.F_BF16_TC if tc else 0, want_nodes=True).cpu().numpy()
    ctx.check()
    want = oracle.build_chi_table_mlp(oracle.Mlp(Ws, bs, oracle.ACT_SILU), nE, nB, lo, hi).chi.astype(np.float64)
    rel = np.abs(got.astype(np.float64) - want) / (np.maximum(want, 1) if not tc else 1 + want)
    _note("node error", rel.max(), 2e-2 if tc else 1e-5)
    assert rel.max() <= (2e-2 if tc else 1e-5)
    # the installed table serves lookups: bilinear interpolation of the nodes the device produced
    E, b = wl.abinitio_pair_batch(seed=9, n=50_000)
    chi = ctx.chi_batch(dev(E), dev(b), 0, 1e-9).cpu().numpy().astype(np.float64)
    tab_g = oracle.ChiTable(got, lo, hi)
    ref = oracle.chi_batch(E, b, 0, 1e-9, table=tab_g)
    sl = _table_slope(tab_g, np.log(E.astype(np.float64)), b.astype(np.float64) / 1e-9)
    assert np.all(np.abs(chi - ref) <= 1e-5 * np.maximum(np.abs(ref), 1) + 2e-4 * sl + 1e-6)
    if not tc:
        # Q23: a network whose output exceeds 64 pi everywhere is capped, node by node
        big = [np.zeros((16, 2), np.float32), np.zeros((1, 16), np.float32)], [np.zeros(16, np.float32), np.array([6.0], np.float32)]
        ctx.set_mlp(1, big[0], big[1], dsmc.ACT_SILU)
        capped = ctx.build_chi_table_mlp(8, 8, lo, hi, want_nodes=True).cpu().numpy()
        assert np.all(capped == np.float32(64 * np.pi))
        with pytest.raises(RuntimeError):
            ctx.build_chi_table_mlp(8, 8, lo, hi, flags=dsmc.F_BF16_TC)  # this shape has no tensor-core image
    ctx.close()


def test_chapman_enskog_from_the_gpu_quadrature(dsmc):
    """(f2) physics check that does not involve the oracle: Omega^(2,2)*(T*) of the LJ gas from the GPU's own
    deflection angles (eqs. 18-19, standard Chapman-Enskog form) against the textbook table."""
    import os
    eps_k, sig = 119.8, 3.405e-10
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "lj_omega22_textbook.txt"))
            if l.strip() and not l.startswith("#")]
    xs, ws = np.polynomial.laguerre.laggauss(20)
    nb, bmax = 2000, 4.0
    bs = (np.arange(nb) + 0.5) * bmax / nb
    ctx = dsmc.Context(1 << 18, 1)
    for Ts, want in ((float(r[0]), float(r[1])) for r in rows):
        E = np.repeat(xs * Ts * eps_k, nb).astype(np.float32)
        b = np.tile(bs * sig, len(xs)).astype(np.float32)
        chi = ctx.chi_exact_batch(dev(E), dev(b), eps_k, sig).cpu().numpy().astype(np.float64).reshape(len(xs), nb)
        q2 = 3.0 * ((1.0 - np.cos(chi) ** 2) * bs[None, :]).sum(axis=1) * bmax / nb
        got = float((ws * xs ** 3 * q2).sum() / 6.0)
        print("Omega22*(T* = %g) = %.4f (textbook %.4f)" % (Ts, got, want))
        assert abs(got / want - 1.0) < 5e-3
    ctx.close()


# --------------------------------------------------------------------------------------- (f1) with replacement
@pytest.mark.parametrize("mode,match", [("table", True), ("table", False), ("mlp", True), ("mlp_tc", True), ("mlp_tc", False)])
def test_collide_abinitio_with_replacement(dsmc, mode, match):
    """pairs drawn with replacement, batch semantics.  Pair indices bit-exact, per-pair g' to the FP32
    tolerance, final velocities to 1e-5 of the thermal scale (the changes of a particle are summed by shared-memory
    atomics in no fixed order), conserved moments to 1e-6 with matching; momentum exact without.  mlp_tc: the chi-MLP
    on the tensor cores (split form on the with-replacement kernels), chi within Q26 of the oracle for every pair and
    every particle within the sum of the allowances of the pairs it sits in."""
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=300_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    tab = _lj_table()
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    ctx.set_mlp(1, Ws, bs, dsmc.ACT_SILU)
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    cm = 0 if mode == "table" else 1
    flags = dsmc.F_PAIR_REPLACE | (dsmc.F_MOMENT_MATCH if match else 0) | (dsmc.F_BF16_TC if mode == "mlp_tc" else 0)
    oflags = oracle.F_PAIR_REPLACE | (oracle.F_MOMENT_MATCH if match else 0)
    prm = dsmc.AbinitioParams(chi_mode=cm, flags=flags)
    oprm = oracle.AbinitioParams(chi_mode=cm, flags=oflags, lnE_min=float(np.float32(prm.lnE_min)), lnE_max=float(np.float32(prm.lnE_max)))
    otab = oracle.ChiTable(tab.chi, float(np.float32(tab.lnE_min)), float(np.float32(tab.lnE_max)))
    v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
    dump = dsmc.PairDump(pop.n, "cuda")
    ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, seed=6, step=1, dump=dump)
    ctx.check()
    ref = oracle.collide_abinitio(cs_h, *v_in, oprm, 6, 1, net=net, table=otab)
    np.testing.assert_array_equal(dump.pair_i.cpu().numpy(), ref.pair_i)
    np.testing.assert_array_equal(dump.pair_j.cpu().numpy(), ref.pair_j)
    sel = ref.pair_i >= 0
    dchi = np.abs(dump.aux.cpu().numpy().astype(np.float64) - ref.aux)
    slope = None
    N = np.diff(cs_h)
    pre = oracle.cell_moments(cs_h, *v_in)
    got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
    ok = N >= 2
    scale = np.repeat(np.sqrt(np.maximum(pre[:, 3], 1e-30) / np.maximum(N, 1)), N)
    allow_v = np.full(pop.n, 1e-5 if mode == "table" else 1e-4)
    if mode == "table":  # Q25 on every pair (oracle-side bound), carried to g' and to the particles of the pair
        idx, bound, gn = _q25_bound(tab, cs_h, v_in, ref, 6, 1)
        assert np.all(dchi[idx] <= bound), "chi outside the Q25 bound: %d pairs" % (dchi[idx] > bound).sum()
        slope = np.zeros_like(dchi)
        slope[idx] = bound
        # a particle moves by (g' - g) / 2 for every pair it sits in: its allowance adds up over those pairs
        kk = np.searchsorted(cs_h, idx, side="right") - 1
        dv = 0.5 * gn * (1e-5 + bound)
        for side in (ref.pair_i, ref.pair_j):
            np.add.at(allow_v, cs_h[kk] + side[idx], 1.05 * dv / scale[cs_h[kk] + side[idx]])
    if mode == "mlp_tc":  # Q26 on every pair from the oracle's chi alone, carried to g' and to the particles
        idx = np.flatnonzero(sel)
        bound = 2e-2 * (1 + np.abs(ref.aux[idx]))
        assert np.all(dchi[idx] <= bound)
        slope = np.zeros_like(dchi)
        slope[idx] = bound
        kk = np.searchsorted(cs_h, idx, side="right") - 1
        gn = np.sqrt(sum((a[cs_h[kk] + ref.pair_i[idx]] - a[cs_h[kk] + ref.pair_j[idx]]) ** 2 for a in v_in))
        dv = 0.5 * gn * (1e-5 + bound)
        for side in (ref.pair_i, ref.pair_j):
            np.add.at(allow_v, cs_h[kk] + side[idx], 1.05 * dv / scale[cs_h[kk] + side[idx]])
        if match:
            # the matching factor alpha = sqrt(Theta_pre / Theta_post) sees the chi differences of ALL pairs of the cell:
            # d(alpha) <= sum_p |c_p| dv_p / Theta with |c_p| <= 4 s and Theta ~ N s^2, and it moves every particle of
            # the cell by d(alpha) |c| <= 16 s mean_p(dv_p / s)  (momentum is exact pair by pair: no shift term)
            pair_part = allow_v - 1e-4
            cell_of = np.repeat(np.arange(len(N)), N)
            mean_part = np.bincount(cell_of, weights=pair_part, minlength=len(N)) / np.maximum(N, 1)
            allow_v = allow_v + 16 * mean_part[cell_of]
    _compare_step(dsmc, ctx, cs, v_in, (vx_s, vy_s, vz_s), dump, ref, 1e-5, 1e-6, slope=slope)
    for a, want in zip((vx_s, vy_s, vz_s), (ref.vx, ref.vy, ref.vz)):
        assert np.all(np.abs(a.cpu().numpy().astype(np.float64) - want) / scale < allow_v)
    assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
    if match:
        assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
    else:
        assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() > 1e-3  # energy is NOT conserved without the correction
    ctx.close()


@pytest.mark.parametrize("tc", [False, True])
def test_collide_vhs_nn_with_replacement(dsmc, tc):
    """SURVEY 8(f1) for the VHS-surrogate operator with NTC acceptance: pairs drawn with replacement, batch
    semantics.  Pair indices and acceptance bit-exact, g' to the FP32 tolerance on the gated set (Q21; tensor cores:
    2e-2), velocities to 1e-4 of the thermal scale, conserved moments to 1e-6."""
    pop = wl.cavity(nx=16, ny=16)
    ctx, net = _setup_vhs(dsmc, pop, 64, 5)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    flags = dsmc.F_NOISE | dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | dsmc.F_ACCEPT | dsmc.F_PAIR_REPLACE
    prm = dsmc.VhsParams(sigma_v=wl.SIGMA_V, flags=flags | (dsmc.F_BF16_TC if tc else 0))
    oprm = oracle.VhsParams(sigma_v=float(np.float32(wl.SIGMA_V)), flags=flags)
    cap = np.full(pop.n_cells, oracle.vhs_sigma_g(6 * wl.SIGMA_V, oprm), np.float32)
    v_in = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
    dump = dsmc.PairDump(pop.n, "cuda")
    ctx.collide_vhs_nn(cs, vx_s, vy_s, vz_s, prm, seed=8, step=4, sigma_cr_max=dev(cap), dump=dump)
    ctx.check()
    ref = oracle.collide_vhs_nn(cs_h, *v_in, net, oprm, 8, 4, sigma_cr_max=cap)
    np.testing.assert_array_equal(dump.pair_i.cpu().numpy(), ref.pair_i)
    np.testing.assert_array_equal(dump.pair_j.cpu().numpy(), ref.pair_j)
    diff = dump.accepted.cpu().numpy() != ref.accepted
    assert diff.sum() <= 2                                   # Q22: decisions within 1e-5 of the threshold
    N = np.diff(cs_h)
    pre = oracle.cell_moments(cs_h, *v_in)
    got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
    ok = N >= 2
    assert (np.linalg.norm(got[ok, :3] - pre[ok, :3], axis=1) / (N[ok] * np.sqrt(pre[ok, 3] / N[ok]))).max() < 1e-6
    assert np.abs(got[ok, 3] / pre[ok, 3] - 1).max() < 1e-6
    sel = ref.pair_i >= 0
    if not diff.any():
        hn = ref.aux
        gate = (hn >= 0.25 * np.median(hn[sel & (ref.accepted == 1)])) | (ref.accepted == 0)
        idx = np.flatnonzero(sel & gate)
        k = np.searchsorted(cs_h, idx, side="right") - 1
        g = np.stack([a[cs_h[k] + ref.pair_i[idx]] - a[cs_h[k] + ref.pair_j[idx]] for a in v_in], axis=1)
        err = np.linalg.norm(dump.gprime.cpu().numpy()[idx].astype(np.float64) - ref.gprime[idx], axis=1) / np.linalg.norm(g, axis=1)
        _note("pair |dg'|/g", err.max(), 2e-2 if tc else 1e-5)
        assert err.max() < (2e-2 if tc else 1e-5)
        scale = np.repeat(np.sqrt(np.maximum(pre[:, 3], 1e-30) / np.maximum(N, 1)), N)
        for a, want in zip((vx_s, vy_s, vz_s), (ref.vx, ref.vy, ref.vz)):
            assert np.median(np.abs(a.cpu().numpy().astype(np.float64) - want) / scale) < (1e-3 if tc else 1e-5)
    multi = np.bincount(np.r_[ref.pair_i[sel] + cs_h[k_all(cs_h, sel)], ref.pair_j[sel] + cs_h[k_all(cs_h, sel)]], minlength=pop.n)
    assert (multi >= 2).mean() > 0.15                         # particles drawn into several pairs of one batch
    ctx.close()


def k_all(cs_h, sel):
    return np.searchsorted(cs_h, np.flatnonzero(sel), side="right") - 1


# --------------------------------------------------------------------------------------- free-running runs (Q20)
@pytest.mark.parametrize("tc", [False, True])
def test_free_running_100_steps_no_artificial_cooling(dsmc, tc):
    """BASELINE.json cfg 1 run freely for 100 steps on the GPU (no re-sync with the oracle, Q20): the cell-wise
    correction must hold every cell's momentum and energy -- "an equilibrium Maxwellian holding its temperature
    without artificial cooling over 100 steps" (north_star) -- while the velocities keep changing."""
    pop = wl.tiny_box()  # 64 cells x 100 particles, 273 K
    ctx, net = _setup_vhs(dsmc, pop, 64, 0)
    vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
    cs_h = cs.cpu().numpy()
    N = np.diff(cs_h)
    v0 = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
    pre = oracle.cell_moments(cs_h, *v0)
    flags = dsmc.F_NOISE | dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | (dsmc.F_BF16_TC if tc else 0)
    prm = dsmc.VhsParams(sigma_v=wl.SIGMA_V, pairs_per_cell=50, flags=flags)
    for step in range(100):
        ctx.collide_vhs_nn(cs, vx_s, vy_s, vz_s, prm, seed=0, step=step)
    ctx.check()
    got = ctx.cell_moments(cs, vx_s, vy_s, vz_s).cpu().numpy()
    drift_e = np.abs(got[:, 3] / pre[:, 3] - 1).max()
    drift_p = (np.linalg.norm(got[:, :3] - pre[:, :3], axis=1) / (N * np.sqrt(pre[:, 3] / N))).max()
    T0 = M * pre[:, 3].sum() / (3 * KB * pop.n)
    T1 = M * got[:, 3].sum() / (3 * KB * pop.n)
    print("100 free steps (tc=%s): max cell energy drift %.2e, momentum drift %.2e, T %.4f -> %.4f K" % (tc, drift_e, drift_p, T0, T1))
    assert drift_e < 1e-5 and drift_p < 1e-5          # 100 steps of <= 1e-6 each, accumulating like a random walk
    assert abs(T1 / T0 - 1) < 1e-6
    moved = np.abs(vx_s.cpu().numpy() - v0[0]) > 1.0
    assert moved.mean() > 0.9                         # the gas did collide
    ctx.close()


def test_relaxation_to_isotropy_with_the_ab_initio_operator(dsmc):
    """Homogeneous relaxation (the paper's relaxation-box setting): a gas whose x-temperature is four
    times its y- and z-temperature relaxes to isotropy under repeated collision steps with the chi table, with the
    total energy of every cell held; a physics-level check of pairing + rotation + matching working together."""
    rng = np.random.default_rng(3)
    n_cells, per = 200, 500
    n = n_cells * per
    sig = math.sqrt(KB * 500.0 / M)
    cell = np.repeat(np.arange(n_cells, dtype=np.int32), per)
    vx = (2.0 * sig * rng.standard_normal(n)).astype(np.float32)
    vy = (1.0 * sig * rng.standard_normal(n)).astype(np.float32)
    vz = (1.0 * sig * rng.standard_normal(n)).astype(np.float32)
    ctx = dsmc.Context(n, n_cells)
    tab = _lj_table()
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    vx_s, vy_s, vz_s, perm, cs = ctx.bin(dev(cell), dev(vx), dev(vy), dev(vz), n_cells)
    e0 = float((vx_s.double() ** 2 + vy_s.double() ** 2 + vz_s.double() ** 2).sum())
    ratio = []
    for step in range(150):
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, dsmc.AbinitioParams(chi_mode=0), seed=5, step=step)
        if step in (0, 9, 149):
            tx = float((vx_s.double() ** 2).mean()); tyz = float(0.5 * ((vy_s.double() ** 2).mean() + (vz_s.double() ** 2).mean()))
            ratio.append(tx / tyz)
    ctx.check()
    e1 = float((vx_s.double() ** 2 + vy_s.double() ** 2 + vz_s.double() ** 2).sum())
    print("T_x / T_yz after 1, 10, 150 steps: %.3f %.3f %.3f (start 4.0)" % tuple(ratio))
    assert ratio[0] < 4.0 and ratio[1] < ratio[0] and abs(ratio[2] - 1.0) < 0.03
    assert abs(e1 / e0 - 1) < 5e-6  # 150 free steps; per step the cells hold their energy to <= 1e-6 (measured drift ~1e-8)
    # relaxed speed distribution is Maxwellian: kurtosis of a component -> 3
    x = vy_s.double().cpu().numpy()
    kurt = float(((x - x.mean()) ** 4).mean() / x.var() ** 2)
    assert abs(kurt - 3.0) < 0.05
    ctx.close()


def test_step_host_equals_the_device_path(dsmc):
    """dsmc_step_host (the end-to-end entry point bench.py times: pinned host buffers in, host buffers out, perm and
    cell_start returned on a side stream under the collide kernels) must give, bit for bit, what dsmc_bin +
    dsmc_collide_abinitio give on device buffers; twice in a row (buffer reuse)."""
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=300_000)
    ctx = dsmc.Context(pop.n, pop.n_cells)
    tab = _lj_table()
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    prm = dsmc.AbinitioParams(chi_mode=0, flags=dsmc.F_MOMENT_MATCH)
    hcell = torch.from_numpy(pop.cell).pin_memory()
    hv = [torch.from_numpy(a).pin_memory() for a in (pop.vx, pop.vy, pop.vz)]
    hout = [torch.empty(pop.n, dtype=torch.float32).pin_memory() for _ in range(3)] + \
           [torch.empty(pop.n, dtype=torch.int32).pin_memory(), torch.empty(pop.n_cells + 1, dtype=torch.int32).pin_memory()]
    for step in (3, 4):
        for t in hout:
            t.fill_(-7)
        ctx.step_host(hcell, *hv, pop.n_cells, hout, abi=prm, seed=9, step=step)
        vx_s, vy_s, vz_s, perm, cs = binned(dsmc, ctx, pop)
        ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, prm, seed=9, step=step)
        ctx.check()
        for got, want in zip(hout, (vx_s, vy_s, vz_s, perm, cs)):
            assert torch.equal(got, want.cpu())
    ctx.close()


def test_step_host_submit_two_contexts_alternating(dsmc):
    """dsmc_step_host_submit (enqueue only) on two contexts, each on its own stream, fed alternately as bench.py's e2e
    loop does: every batch gives, bit for bit, what the synchronous dsmc_step_host gives for the same (input, step)."""
    pops = [wl.mach10_cylinder(seed=s, nx=60, ny=30, n_total=300_000) for s in (4, 5)]
    tab = _lj_table()
    prm = dsmc.AbinitioParams(chi_mode=0, flags=dsmc.F_MOMENT_MATCH)
    ctxs, streams = [], []
    for _ in range(2):
        c = dsmc.Context(pops[0].n, pops[0].n_cells)
        c.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
        ctxs.append(c)
        streams.append(torch.cuda.Stream())
    ref = dsmc.Context(pops[0].n, pops[0].n_cells)
    ref.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)

    def host_in(pop):
        return [torch.from_numpy(a).pin_memory() for a in (pop.cell, pop.vx, pop.vy, pop.vz)]

    def host_out(pop):
        return [torch.empty(pop.n, dtype=torch.float32).pin_memory() for _ in range(3)] + \
               [torch.empty(pop.n, dtype=torch.int32).pin_memory(), torch.empty(pop.n_cells + 1, dtype=torch.int32).pin_memory()]

    hin = [host_in(p) for p in pops]
    houts = [host_out(pops[0]) for _ in range(2)]
    want = host_out(pops[0])
    torch.cuda.synchronize()
    results = []
    for t in range(6):
        k = t & 1
        if t >= 2:  # the lane's previous batch must be complete before its buffers are reused
            ctxs[k].check()
            results.append((t - 2, [x.clone() for x in houts[k]]))
        with torch.cuda.stream(streams[k]):
            ctxs[k].step_host(*hin[(t // 2) & 1], pops[0].n_cells, houts[k], abi=prm, seed=9, step=t, submit_only=True)
    for k in (0, 1):
        ctxs[k].check()
        results.append((4 + k, [x.clone() for x in houts[k]]))
    assert sorted(t for t, _ in results) == list(range(6))
    for t, got in results:
        ref.step_host(*hin[(t // 2) & 1], pops[0].n_cells, want, abi=prm, seed=9, step=t)
        for g, w in zip(got, want):
            assert torch.equal(g, w), "batch %d differs" % t
    for c in ctxs + [ref]:
        c.close()

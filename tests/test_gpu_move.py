"""GPU parity tests (-m gpu) of the minimal DSMC loop around the collision step: free flight +
Maxwell walls (dsmc_move_couette), the gather into sorted order, the per-cell sampling sums and the device-side
loop (dsmc_couette_run), against the CPU oracle on the same seeded inputs.

Decisions taken in floating point (wall hit, diffuse or specular, cell index) are compared wherever the oracle
reports a margin above the FP32 resolution (1e-5 of the gap); elsewhere either answer is right and the test checks
that the GPU's own outputs are consistent (position inside the gap, cell = floor(x n_cells / L))."""
import math

import numpy as np
import pytest

import oracle
from paper_2602_21244_b200 import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

RT = 208.13 * 273.0


@pytest.fixture(scope="module")
def dsmc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2602_21244_b200 import dsmc as mod
    return mod


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gas(n, seed, L, rt=RT):
    rng = np.random.default_rng(seed)
    x = (rng.random(n) * L).astype(np.float32)
    v = rng.normal(0.0, math.sqrt(rt), (3, n)).astype(np.float32)
    return np.minimum(x, np.float32(L)), v


@pytest.mark.parametrize("case", ["typical", "many_bounces", "specular", "empty"])
def test_move_couette_matches_oracle(dsmc, case):
    L, K, U = 0.05, 200, 500.0
    n = 300_007
    dt = 0.5 * (L / K) / math.sqrt(RT)
    acc = 0.8
    if case == "many_bounces":
        dt = 0.9 * L / math.sqrt(RT)  # a thermal particle crosses the gap in a step: up to > DSMC_MAX_BOUNCES hits
    if case == "specular":
        acc, dt = 0.0, 0.4 * L / math.sqrt(RT)
    if case == "empty":
        n = 0
    x, v = _gas(n, 3, L)
    geo_o = oracle.CouetteParams(float(np.float32(L)), float(np.float32(dt)), U, float(np.float32(RT)),
                                 float(np.float32(acc)), K)
    geo = dsmc.CouetteParams(L, dt, U, RT, acc, K)
    ctx = dsmc.Context(max(n, 1), K)
    xd, vxd, vyd, vzd = dev(x), dev(v[0]), dev(v[1]), dev(v[2])
    nb_d = torch.zeros(n, dtype=torch.int32, device="cuda")
    cell_d = ctx.move_couette(xd, vxd, vyd, vzd, geo, seed=77, step=5, bounces=nb_d)
    ctx.check()
    if n == 0:
        ctx.close()
        return
    xo, vxo, vyo, vzo, cell_o, nb_o, mg = oracle.move_couette(x, v[0], v[1], v[2], geo_o, 77, 5)
    xg, vxg, vyg, vzg = (t.cpu().numpy() for t in (xd, vxd, vyd, vzd))
    cell_g, nb_g = cell_d.cpu().numpy(), nb_d.cpu().numpy()
    # validity, every particle
    Lf = np.float32(L)
    assert np.all((xg >= 0) & (xg <= Lf))
    cpl = np.float32(K / float(Lf))
    assert np.array_equal(cell_g, np.clip(np.floor(xg * cpl).astype(np.int64), 0, K - 1))
    # decisions and values where the oracle's decisions are resolvable in FP32
    sure = mg > 1e-5
    print("%s: %.4f%% of particles within 1e-5 of a decision threshold; bounces up to %d; %.1f%% hit a wall"
          % (case, 100 * (1 - sure.mean()), nb_o.max(), 100 * (nb_o > 0).mean()))
    assert sure.mean() > 0.995
    assert np.array_equal(nb_g[sure], nb_o[sure])
    assert np.array_equal(cell_g[sure], cell_o[sure])
    assert np.abs(xg[sure] - xo[sure]).max() <= 4e-6 * L
    for got, want, raw in ((vxg, vxo, v[0]), (vyg, vyo, v[1]), (vzg, vzo, v[2])):
        assert np.abs(got[sure] - want[sure]).max() <= 2e-5 * math.sqrt(RT + U * U)
        untouched = sure & (nb_o == 0)
        assert np.array_equal(got[untouched], raw[untouched])  # bit-exact where no wall was met
    if case == "many_bounces":
        assert nb_o.max() == oracle.MAX_BOUNCES and (nb_o >= 2).mean() > 0.05
    if case == "specular":
        assert np.array_equal(vyg, v[1]) and np.array_equal(vzg, v[2])
    ctx.close()


def test_gather_bit_exact(dsmc):
    rng = np.random.default_rng(1)
    n = 200_003
    perm = rng.permutation(n).astype(np.int32)
    src = rng.normal(size=n).astype(np.float32)
    ctx = dsmc.Context(n, 1)
    got = ctx.gather_f32(dev(perm), dev(src)).cpu().numpy()
    ctx.check()
    assert np.array_equal(got, src[perm])
    ctx.close()


def test_sample_cells_matches_oracle_and_accumulates(dsmc):
    pop = wl.mach10_cylinder(nx=60, ny=30, n_total=200_000)  # ragged cells, some empty, some large
    ctx = dsmc.Context(pop.n, pop.n_cells)
    vx_s, vy_s, vz_s, perm, cs = ctx.bin(dev(pop.cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), pop.n_cells)
    acc = torch.zeros((pop.n_cells, 8), dtype=torch.float64, device="cuda")
    ctx.sample_cells(cs, vx_s, vy_s, vz_s, acc)
    ctx.check()
    cs_h = cs.cpu().numpy()
    v = [t.cpu().numpy().astype(np.float64) for t in (vx_s, vy_s, vz_s)]
    want = oracle.sample_cells(cs_h, *v)
    got = acc.cpu().numpy()
    assert np.array_equal(got[:, 0], want[:, 0])
    scale = np.maximum(want[:, 4:7].sum(axis=1, keepdims=True), 1.0)  # sum of squares bounds every term
    assert np.abs(got - want).max() <= 1e-12 * scale.max()
    assert (np.abs(got - want) / scale).max() <= 1e-13
    ctx.sample_cells(cs, vx_s, vy_s, vz_s, acc)
    ctx.check()
    assert np.allclose(acc.cpu().numpy(), 2 * want, rtol=1e-13, atol=1e-9)
    ctx.close()


def _lj_table(nE=128, nB=128):
    return oracle.build_chi_table(oracle.lj_argon(), nE, nB, n_panels=2)


def test_couette_run_equals_the_staged_calls(dsmc):
    """dsmc_couette_run is plumbing: three steps of it must give, bit for bit, what the individual entry points give
    when called in the same order (move -> bin -> gather -> collide -> sample)."""
    L, K, U = 0.02, 64, 500.0
    n = 64 * 300 + 11
    dt = 0.5 * (L / K) / math.sqrt(RT)
    x, v = _gas(n, 8, L)
    geo = dsmc.CouetteParams(L, dt, U, RT, 1.0, K)
    prm = dsmc.AbinitioParams(pairs_per_cell=40, flags=dsmc.F_MOMENT_MATCH)
    tab = _lj_table(64, 64)
    ctx = dsmc.Context(n, K)
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    # staged
    xs, vxs, vys, vzs = dev(x), dev(v[0]), dev(v[1]), dev(v[2])
    acc_s = torch.zeros((K, 8), dtype=torch.float64, device="cuda")
    for k in range(3):
        cell = ctx.move_couette(xs, vxs, vys, vzs, geo, seed=5, step=10 + k)
        vxs, vys, vzs, perm, cs = ctx.bin(cell, vxs, vys, vzs, K)
        xs = ctx.gather_f32(perm, xs)
        ctx.collide_abinitio(cs, vxs, vys, vzs, prm, seed=5, step=10 + k)
        if k >= 1:
            ctx.sample_cells(cs, vxs, vys, vzs, acc_s)
    ctx.check()
    # one call
    xr, vxr, vyr, vzr = dev(x), dev(v[0]), dev(v[1]), dev(v[2])
    acc_r = torch.zeros((K, 8), dtype=torch.float64, device="cuda")
    ctx.couette_run(xr, vxr, vyr, vzr, geo, 3, abi=prm, seed=5, step0=10, sample_from=1, acc=acc_r)
    for a, b in ((xs, xr), (vxs, vxr), (vys, vyr), (vzs, vzr), (acc_s, acc_r)):
        assert torch.equal(a, b)
    assert float(acc_r[:, 0].sum()) == 2 * n
    ctx.close()


def test_couette_flow_profiles_against_the_oracle_loop(dsmc):
    """A physical run (P:L183-187 setting in miniature): gas between diffuse walls moving at +-U, ab initio table
    operator with a fixed number of collision pairs per cell and step.  The GPU loop and the oracle loop (same
    stages, FP64) are chaotic, so they are compared through their time-averaged profiles: wall-parallel velocity
    u_y(x), shear stress <vx vy> and temperature.  Physics checks on the GPU result: the shear stress is uniform
    across the gap (momentum conservation), below the free-molecular value U sqrt(2RT/pi), the velocity profile is
    antisymmetric with slip at the walls (|u| < U), viscous heating raises T above the wall temperature."""
    L, K, U = 0.02, 20, 500.0
    per = 400
    n = K * per
    dt = 0.4 * (L / K) / math.sqrt(RT)
    n_steps, sample_from = 500, 250
    x, v = _gas(n, 12, L)
    geo = dsmc.CouetteParams(L, dt, U, RT, 1.0, K)
    geo_o = oracle.CouetteParams(float(np.float32(L)), float(np.float32(dt)), U, float(np.float32(RT)), 1.0, K)
    m_pairs = 60
    tab = _lj_table(64, 64)
    ctx = dsmc.Context(n, K)
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    prm = dsmc.AbinitioParams(pairs_per_cell=m_pairs, flags=dsmc.F_MOMENT_MATCH)
    xd, vxd, vyd, vzd = dev(x), dev(v[0]), dev(v[1]), dev(v[2])
    acc = torch.zeros((K, 8), dtype=torch.float64, device="cuda")
    ctx.couette_run(xd, vxd, vyd, vzd, geo, n_steps, abi=prm, seed=1, step0=0, sample_from=sample_from, acc=acc)
    G = acc.cpu().numpy()
    # oracle loop
    prm_o = oracle.AbinitioParams(pairs_per_cell=m_pairs, flags=oracle.F_MOMENT_MATCH)
    xo = x.astype(np.float64)
    vo = [a.astype(np.float64) for a in v]
    O = np.zeros((K, 8))
    for k in range(n_steps):
        xo, vo[0], vo[1], vo[2], cell, nb, mg = oracle.move_couette(xo, vo[0], vo[1], vo[2], geo_o, 1, k)
        rc, perm, cs = oracle.bin_particles(cell, K)
        xo = xo[perm]
        vo = [a[perm] for a in vo]
        res = oracle.collide_abinitio(cs, vo[0], vo[1], vo[2], prm_o, 1, k, table=tab)
        vo = [res.vx, res.vy, res.vz]
        if k >= sample_from:
            oracle.sample_cells(cs, vo[0], vo[1], vo[2], O)

    def fields(A):
        cnt = A[:, 0]
        uy = A[:, 2] / cnt
        txy = (A[:, 7] - A[:, 1] * uy) / cnt.mean()   # momentum flux per mean density: n <c_x c_y> / n_0
        T = ((A[:, 4] + A[:, 5] + A[:, 6]) / cnt - (A[:, 1] ** 2 + A[:, 2] ** 2 + A[:, 3] ** 2) / cnt ** 2) / 3.0
        return cnt, uy, txy, T

    cg, uyg, tg, Tg = fields(G)
    co, uyo, to, To = fields(O)
    fm = U * math.sqrt(2 * RT / math.pi)
    print("Couette loop: u_y(wall cells) GPU %.1f / %.1f, oracle %.1f / %.1f; <vx vy> GPU %.0f oracle %.0f "
          "(free-molecular %.0f); T/T_w GPU %.3f oracle %.3f"
          % (uyg[0], uyg[-1], uyo[0], uyo[-1], tg.mean(), to.mean(), -fm, Tg.mean() / RT, To.mean() / RT))
    assert cg.sum() == co.sum() == (n_steps - sample_from) * n
    assert np.abs(cg / cg.sum() - 1.0 / K).max() < 0.1 / K and np.abs(co / co.sum() - 1.0 / K).max() < 0.1 / K
    assert np.abs(uyg - uyo).max() < 0.05 * U             # profiles agree within the statistical scatter
    assert abs(tg.mean() / to.mean() - 1) < 0.04
    assert abs(Tg.mean() / To.mean() - 1) < 0.03
    # physics of the GPU result
    assert np.abs(tg / tg.mean() - 1).max() < 0.06        # uniform momentum flux
    assert -fm < tg.mean() < -0.2 * fm
    assert np.all(np.diff(uyg[2:-2]) > -0.05 * U) and uyg[0] < -0.3 * U and uyg[-1] > 0.3 * U
    assert abs(uyg[0]) < U and abs(uyg[-1]) < U           # velocity slip
    assert np.abs(uyg + uyg[::-1]).max() < 0.06 * U       # antisymmetry
    assert Tg.mean() > 1.02 * RT                          # viscous heating
    ctx.close()


# ------------------------------------------------------------------ f1: NTC candidate counts (Q31)
def test_ntc_counts_bit_exact_and_per_cell_requests(dsmc):
    """dsmc_ntc_counts against the oracle over several steps (counts and FP64 remainders bit-exact), then one fused
    step of each operator driven by the per-cell counts: pair indices bit-exact against the oracle, every cell ran
    min(count, N/2) pairs."""
    rng = np.random.default_rng(4)
    counts = rng.integers(0, 120, 900)
    counts[3], counts[4], counts[5], counts[6] = 0, 1, 2, 2048
    pop = wl._populate("ragged", counts, np.full(900, 300.0), np.zeros(900), np.zeros(900), 4)
    K = pop.n_cells
    ctx = dsmc.Context(pop.n, K)
    vx_s, vy_s, vz_s, perm, cs = ctx.bin(dev(pop.cell), dev(pop.vx), dev(pop.vy), dev(pop.vz), K)
    cs_h = cs.cpu().numpy()
    cap = (rng.random(K) * 2e-16 + 1e-16).astype(np.float32)
    coef = 0.37 / (60 * float(cap.mean()))     # about 0.37 N candidates in a 120-particle cell
    R_o = np.zeros(K)
    R_d = torch.zeros(K, dtype=torch.float64, device="cuda")
    cap_d = dev(cap)
    for t in range(5):
        want = oracle.ntc_counts(cs_h, cap, coef, R_o)
        got = ctx.ntc_counts(cs, cap_d, coef, R_d)
        ctx.check()
        assert np.array_equal(got.cpu().numpy(), want)
        assert np.array_equal(R_d.cpu().numpy(), R_o)
    assert want.max() > 60 and (want == 0).sum() > 3 and want[6] > 1024   # some above N/2, some zero
    N = np.diff(cs_h)
    M_want = np.where(N >= 2, np.minimum(want, N // 2), 0)
    # ab initio table operator with the per-cell counts
    tab = _lj_table(64, 64)
    ctx.set_chi_table(tab.chi, tab.lnE_min, tab.lnE_max)
    v_in = [a.cpu().numpy().astype(np.float64) for a in (vx_s, vy_s, vz_s)]
    dump = dsmc.PairDump(pop.n, "cuda")
    ctx.collide_abinitio(cs, vx_s, vy_s, vz_s, dsmc.AbinitioParams(pairs_count=got), seed=9, step=1, dump=dump)
    ctx.check()
    ref = oracle.collide_abinitio(cs_h, *v_in, oracle.AbinitioParams(pairs_count=want), 9, 1, table=tab)
    pi = dump.pair_i.cpu().numpy()
    assert np.array_equal(pi, ref.pair_i) and np.array_equal(dump.pair_j.cpu().numpy(), ref.pair_j)
    per_cell = np.add.reduceat((pi >= 0).astype(np.int64), cs_h[:-1][N > 0])
    assert np.array_equal(per_cell, M_want[N > 0])
    for a, w in zip((vx_s, vy_s, vz_s), (ref.vx, ref.vy, ref.vz)):
        assert np.abs(a.cpu().numpy() - w).max() < 2e-4 * 400
    # VHS-NN with NTC acceptance on the same counts
    Ws, bs = wl.random_mlp(2, [8, 64, 64, 3])
    ctx.set_mlp(0, Ws, bs, dsmc.ACT_TANH)
    net = oracle.Mlp(Ws, bs, oracle.ACT_TANH)
    flags = dsmc.F_NOISE | dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | dsmc.F_ACCEPT
    oprm = oracle.VhsParams(sigma_v=float(np.float32(wl.SIGMA_V)), flags=flags, pairs_count=want)
    cap_v = np.full(K, oracle.vhs_sigma_g(6 * wl.SIGMA_V, oprm), np.float32)
    v_in = [a.cpu().numpy().astype(np.float64) for a in (vx_s, vy_s, vz_s)]
    dump = dsmc.PairDump(pop.n, "cuda")
    ctx.collide_vhs_nn(cs, vx_s, vy_s, vz_s, dsmc.VhsParams(sigma_v=wl.SIGMA_V, flags=flags, pairs_count=got),
                       seed=9, step=2, sigma_cr_max=dev(cap_v), dump=dump)
    ctx.check()
    ref = oracle.collide_vhs_nn(cs_h, *v_in, net, oprm, 9, 2, sigma_cr_max=cap_v)
    assert np.array_equal(dump.pair_i.cpu().numpy(), ref.pair_i)
    assert np.array_equal(dump.pair_j.cpu().numpy(), ref.pair_j)
    assert (dump.accepted.cpu().numpy() != ref.accepted).sum() <= 2      # Q22: decisions at the threshold
    ctx.close()


def test_couette_viscosity_matches_chapman_enskog(dsmc):
    """End-to-end physics of the whole device-side loop with NTC rate control and the ab initio table
    operator: argon (LJ 12-6) between diffuse walls at Kn = 0.05.  In the bulk the momentum flux must equal
    mu(T) du_y/dx with the Chapman-Enskog viscosity of the SAME potential, mu = 5/16 sqrt(pi m k T) / (pi sigma^2
    Omega22*(T*)) (the paper's eqs. 17-19 in standard form, Q28), Omega22* evaluated here from the oracle's
    deflection angles (pinned to the textbook table by P14).  Nothing in the collision path knows about viscosity:
    pairing, NTC counts, acceptance, the chi table, the rotation and the cell-wise matching all have to be right
    for this number to come out."""
    KB, m = 1.380649e-23, 6.63e-26
    eps_k, sig = 119.8, 3.405e-10
    Tw, U = 273.0, 150.0
    rt = KB * Tw / m
    b_max = 1.0e-9
    n_dens = 1.0e20
    K, per = 60, 150
    L = 0.345                                   # Kn = 0.05 on the viscosity-based mean free path (17 mm)
    dt = 1.0e-6
    g_max = 2000.0
    sigma_T = math.pi * b_max ** 2
    geo = dsmc.CouetteParams(L, dt, U, rt, 1.0, K, ntc_coef=n_dens * dt / per, sigma_cr_max=sigma_T * g_max)
    n = K * per
    rng = np.random.default_rng(31)
    x = (rng.random(n) * L).astype(np.float32)
    v = rng.normal(0.0, math.sqrt(rt), (3, n))
    v[1] += 0.85 * U * (2 * x / L - 1)          # start near the steady shear profile: short transient
    v = v.astype(np.float32)
    ctx = dsmc.Context(n, K)
    ctx.build_chi_table_lj(512, 512, b_max=b_max, eps_over_k=eps_k, sigma=sig)
    prm = dsmc.AbinitioParams(mass=m, b_max=b_max, flags=dsmc.F_MOMENT_MATCH | dsmc.F_ACCEPT)
    xd, vxd, vyd, vzd = dev(x), dev(v[0]), dev(v[1]), dev(v[2])
    acc = torch.zeros((K, 8), dtype=torch.float64, device="cuda")
    n_steps, sample_from = 30000, 6000
    ctx.couette_run(xd, vxd, vyd, vzd, geo, n_steps, abi=prm, seed=2, step0=0, sample_from=sample_from, acc=acc)
    A = acc.cpu().numpy()
    cnt = A[:, 0]
    uy = A[:, 2] / cnt
    flux = (A[:, 7] - A[:, 1] * uy).sum() / cnt.sum()            # <n c_x c_y> / n_0, uniform across the gap
    T = m * ((A[:, 4] + A[:, 5] + A[:, 6]) / cnt - (A[:, 1] ** 2 + A[:, 2] ** 2 + A[:, 3] ** 2) / cnt ** 2) / (3 * KB)
    xc = (np.arange(K) + 0.5) * L / K
    bulk = slice(10, K - 10)                                     # outside the Knudsen layers (3 mean free paths)
    slope = np.polyfit(xc[bulk], uy[bulk], 1)[0]
    rho0 = n_dens * m
    mu_meas = -rho0 * flux / slope
    T_bulk = T[bulk].mean()
    # Chapman-Enskog viscosity of LJ argon at T_bulk from the oracle's deflection angles
    pot = oracle.lj_argon()
    xs, ws = np.polynomial.laguerre.laggauss(20)
    nb, bm = 400, 4.0
    bs = (np.arange(nb) + 0.5) * bm / nb

    def q2_star(Es):
        chi = np.array([oracle.chi_exact(pot, Es * eps_k * KB, b * sig) for b in bs])
        return 3.0 * np.sum((1.0 - np.cos(chi) ** 2) * bs) * bm / nb

    Ts = T_bulk / eps_k
    omega = sum(w * xx ** 3 * q2_star(xx * Ts) for xx, w in zip(xs, ws)) / 6.0
    mu_ce = 5.0 / 16.0 * math.sqrt(math.pi * m * KB * T_bulk) / (math.pi * sig ** 2 * omega)
    print("Couette, LJ argon, Kn 0.05: mu = %.4e Pa s measured, %.4e Chapman-Enskog (Omega22* = %.4f at T = %.1f K);"
          " slope %.1f 1/s of %.1f no-slip; T_max %.1f K" % (mu_meas, mu_ce, omega, T_bulk, slope, 2 * U / L, T.max()))
    assert 0.75 * 2 * U / L < slope < 2 * U / L                  # velocity slip
    assert Tw < T_bulk < Tw + 20 and T.argmax() in range(K // 2 - 12, K // 2 + 12)   # viscous heating, centred
    assert abs(mu_meas / mu_ce - 1) < 0.06
    ctx.close()


def test_argument_errors_of_the_loop_entry_points(dsmc):
    """Host-detectable errors return DSMC_ERR_INVALID_ARG and launch nothing; a chi table with a non-finite node is
    refused (Q23: such a node would turn every pair near it, and through the matching its whole cell, into NaN)."""
    ctx = dsmc.Context(1024, 8)
    x = torch.zeros(16, device="cuda")
    v = [torch.zeros(16, device="cuda") for _ in range(3)]
    good = dict(L=1.0, dt=1e-3, u_wall=1.0, rt_wall=1.0, accommodation=1.0, n_cells=8)
    l0 = ctx.launch_count()
    for bad in (dict(L=0.0), dict(rt_wall=0.0), dict(accommodation=1.5), dict(accommodation=-0.1), dict(n_cells=0)):
        with pytest.raises(dsmc.DsmcError) as e:
            ctx.move_couette(x, *v, dsmc.CouetteParams(**{**good, **bad}), seed=0, step=0)
        assert e.value.status == -1
    with pytest.raises(dsmc.DsmcError):   # n_cells above the context's capacity
        ctx.couette_run(x, *v, dsmc.CouetteParams(**{**good, "n_cells": 9}), 1, abi=dsmc.AbinitioParams())
    with pytest.raises(dsmc.DsmcError):   # neither operator
        ctx.couette_run(x, *v, dsmc.CouetteParams(**good), 1)
    with pytest.raises(dsmc.DsmcError):   # NTC without a bound
        ctx.build_chi_table_lj(16, 16)
        ctx.couette_run(x, *v, dsmc.CouetteParams(**{**good, "ntc_coef": 1.0}), 1, abi=dsmc.AbinitioParams())
    assert ctx.launch_count() - l0 <= 2   # only the table build launched anything
    tab = np.ones((8, 8), np.float32)
    tab[3, 4] = np.inf
    with pytest.raises(dsmc.DsmcError) as e:
        ctx.set_chi_table(tab, math.log(5.0), math.log(6e4))
    assert e.value.status == -1
    tab[3, 4] = np.nan
    with pytest.raises(dsmc.DsmcError):
        ctx.set_chi_table(tab, math.log(5.0), math.log(6e4))
    ctx.close()

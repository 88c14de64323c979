"""Pins for the CPU oracle (-m "not gpu").  Each test checks the oracle against something other
than itself: values printed in the paper / known-answer vectors (tests/golden/), closed forms,
invariants the paper states as exact, library routines on special cases, brute force on tiny
inputs.  Pin numbers P1..P13 follow SURVEY.md section 8(c) / DESIGN.md."""
import math
import os

import numpy as np
import pytest
from scipy import integrate, optimize, special, stats

import oracle
from paper_2602_21244_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M = wl.MASS_AR
KB = 1.380649e-23


# ------------------------------------------------------------------------------------ P1 Philox
def test_p1_philox_known_answers():
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert oracle.philox4x32_10(w[0:4], w[4:6]) == w[6:10]


def test_u01_is_open_interval_and_exact_in_fp32():
    assert oracle.u01(0) == 0.5 / 2**23
    assert oracle.u01(0xFFFFFFFF) == 1.0 - 0.5 / 2**23
    for x in (0, 511, 512, 0x80000000, 0xFFFFFFFF, 123456789, 0xFFFFFE00):
        u = oracle.u01(x)
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u


def test_rng_addressing_streams_are_distinct_and_keyed():
    seed = 0x1234567899
    r0 = oracle.philox4x32_10([5 >> 2, 7, 3, 0], [seed & 0xFFFFFFFF, seed >> 32])
    assert oracle.pair_key(seed, 3, 7, 5) == r0[5 & 3]
    # pair 9: (U_b, U_eps) = words 2, 3 of stream-1 block 9 >> 1; U_acc = word 9 & 3 of stream-3 block 9 >> 2
    r1 = oracle.philox4x32_10([9 >> 1, 7, 3, 1], [seed & 0xFFFFFFFF, seed >> 32])
    r3 = oracle.philox4x32_10([9 >> 2, 7, 3, 3], [seed & 0xFFFFFFFF, seed >> 32])
    np.testing.assert_array_equal(oracle.pair_uniforms(seed, 3, 7, 9), [oracle.u01(x) for x in (r3[9 & 3], r1[2], r1[3])])
    r1e = oracle.philox4x32_10([8 >> 1, 7, 3, 1], [seed & 0xFFFFFFFF, seed >> 32])
    np.testing.assert_array_equal(oracle.pair_uniforms(seed, 3, 7, 8)[1:], [oracle.u01(x) for x in (r1e[0], r1e[1])])
    # normals: Box-Muller identity xi0^2 + xi1^2 = -2 ln u0
    r2 = oracle.philox4x32_10([9, 7, 3, 2], [seed & 0xFFFFFFFF, seed >> 32])
    xi = oracle.pair_normals(seed, 3, 7, 9)
    assert abs(xi[0] ** 2 + xi[1] ** 2 + 2 * math.log(oracle.u01(r2[0]))) < 1e-12


def test_normals_are_standard_gaussian():
    xi = np.array([oracle.pair_normals(42, 1, c, s) for c in range(20) for s in range(500)])
    for a in range(3):
        assert stats.kstest(xi[:, a], "norm").pvalue > 1e-3
    assert np.abs(np.corrcoef(xi.T) - np.eye(3)).max() < 0.05


# ------------------------------------------------------------------------------------ a1 binning
def test_bin_is_the_stable_sort_by_cell():
    rng = np.random.default_rng(0)
    cell = rng.integers(0, 37, 5000).astype(np.int32)
    rc, perm, cs = oracle.bin_particles(cell, 37)
    assert rc == 0
    np.testing.assert_array_equal(perm, np.argsort(cell, kind="stable"))
    np.testing.assert_array_equal(cs, np.concatenate([[0], np.cumsum(np.bincount(cell, minlength=37))]))
    rc, _, _ = oracle.bin_particles(np.array([0, 37], np.int32), 37)
    assert rc == -2
    rc, perm, cs = oracle.bin_particles(np.zeros(0, np.int32), 4)
    assert rc == 0 and cs.tolist() == [0, 0, 0, 0, 0]


# ------------------------------------------------------------------------------------ a2 moments
def test_cell_moments_and_state_against_numpy_statistics():
    rng = np.random.default_rng(1)
    cs = np.array([0, 10, 10, 11, 300], np.int32)
    v = rng.normal(100.0, 300.0, (3, 300))
    mom = oracle.cell_moments(cs, *v)
    for k in range(4):
        seg = v[:, cs[k]:cs[k + 1]]
        np.testing.assert_allclose(mom[k, :3], seg.sum(axis=1), rtol=1e-13, atol=1e-9)
        np.testing.assert_allclose(mom[k, 3], (seg ** 2).sum(), rtol=1e-13)
    ubar, theta, T = oracle.cell_state(*v, M)
    np.testing.assert_allclose(ubar, v.mean(axis=1), rtol=1e-13)
    np.testing.assert_allclose(theta, 300 * np.var(v, axis=1).sum(), rtol=1e-12)
    np.testing.assert_allclose(T, M * np.var(v, axis=1).sum() / (3 * KB), rtol=1e-12)


def test_p12_maxwellian_temperature_and_mean_speed():
    """eq. 12: <v> = sqrt(8 kB T / (pi m)); paper prints 380.2270 m/s at 272.78 K."""
    gold = dict(l.split() for l in open(os.path.join(GOLD, "paper_printed_values.txt")) if not l.startswith("#"))
    T0 = float(gold["mean_speed_T"])
    closed = math.sqrt(8 * KB * T0 / (math.pi * M))
    assert abs(closed / float(gold["mean_speed_value"]) - 1) < 5e-4  # loose: constants differ (Q18)
    pop = wl.tiny_box(seed=5, n_cells=1, per_cell=400000, T=T0)
    _, _, T = oracle.cell_state(pop.vx, pop.vy, pop.vz, M)
    assert abs(T / T0 - 1) < 5e-3
    speed = np.sqrt(pop.vx.astype(np.float64) ** 2 + pop.vy.astype(np.float64) ** 2 + pop.vz.astype(np.float64) ** 2)
    assert abs(speed.mean() / closed - 1) < 3e-3


# ------------------------------------------------------------------------------------ a3 pairing
def test_p11_pairing_brute_force_tiny_cells():
    M2, pi = oracle.pairing(1, 0, 0, 2)
    assert M2 == 1 and sorted(pi.tolist()) == [0, 1]
    assert oracle.pairing(1, 0, 0, 1)[0] == 0 and oracle.pairing(1, 0, 0, 0)[0] == 0
    # N = 3: one of three pairs + a spectator, each with frequency 1/3
    cnt = {}
    trials = 9000
    for c in range(trials):
        Mk, pi = oracle.pairing(7, 2, c, 3)
        assert Mk == 1 and sorted(pi.tolist()) == [0, 1, 2]
        key = tuple(sorted(pi[:2].tolist()))
        cnt[key] = cnt.get(key, 0) + 1
    assert len(cnt) == 3
    for v in cnt.values():
        assert abs(v - trials / 3) < 4 * math.sqrt(trials * 2 / 9)
    # N = 4: three perfect matchings, each 1/3
    cnt = {}
    for c in range(trials):
        Mk, pi = oracle.pairing(11, c % 5, c, 4)
        assert Mk == 2
        m = tuple(sorted([tuple(sorted(pi[0:2].tolist())), tuple(sorted(pi[2:4].tolist()))]))
        cnt[m] = cnt.get(m, 0) + 1
    assert len(cnt) == 3
    for v in cnt.values():
        assert abs(v - trials / 3) < 4 * math.sqrt(trials * 2 / 9)


def test_pairing_is_argsort_of_keys_and_respects_request():
    N = 101
    Mk, pi = oracle.pairing(99, 4, 17, N, 30)
    assert Mk == 30
    keys = np.array([oracle.pair_key(99, 4, 17, p) for p in range(N)], np.uint64)
    np.testing.assert_array_equal(pi, np.lexsort((np.arange(N), keys)))
    assert oracle.pairing(99, 4, 17, N, 80)[0] == 50
    assert oracle.pairing(99, 4, 17, N, -1)[0] == 50


def test_each_particle_is_equally_likely_to_be_left_out_or_first():
    N, trials = 5, 10000
    last = np.zeros(N)
    for c in range(trials):
        last[oracle.pairing(3, 0, c, N)[1][-1]] += 1
    assert np.all(np.abs(last - trials / N) < 4.5 * math.sqrt(trials * (1 / N) * (1 - 1 / N)))


# ------------------------------------------------------------------------------------ MLP
def test_mlp_closed_form_cases():
    # non-square, asymmetric weights: a transposed operand or dropped bias changes the answer
    W1 = np.array([[1, 2], [3, 4], [5, 6]], np.float32)
    net = oracle.Mlp([W1, np.eye(3, dtype=np.float32)], [np.array([0.5, -100, 0], np.float32), np.array([1, 2, 3], np.float32)], oracle.ACT_RELU)
    np.testing.assert_allclose(oracle.mlp_forward(net, [1.0, 10.0]), [21.5 + 1, 0 + 2, 65 + 3])
    net.act = oracle.ACT_TANH
    np.testing.assert_allclose(oracle.mlp_forward(net, [0.01, 0.02]), [math.tanh(0.55) + 1, math.tanh(-99.89) + 2, math.tanh(0.17) + 3], rtol=1e-14)
    net.act = oracle.ACT_SILU
    np.testing.assert_allclose(oracle.mlp_forward(net, [0.5, 0.0])[0], 1.0 / (1 + math.exp(-1.0)) + 1, rtol=1e-14)
    # |x| = relu(x) + relu(-x), three layers
    net = oracle.Mlp([np.array([[1], [-1]], np.float32), np.array([[1, 1]], np.float32), np.array([[2]], np.float32)],
                     [np.zeros(2, np.float32), np.zeros(1, np.float32), np.array([1], np.float32)], oracle.ACT_RELU)
    for x in (-3.0, 0.25):
        np.testing.assert_allclose(oracle.mlp_forward(net, [x]), [2 * abs(x) + 1])


def _probe_net(n_in, feats):
    """ReLU network whose 3 outputs are input features feats[0..2]: out = relu(x) - relu(-x)."""
    W1 = np.zeros((6, n_in), np.float32)
    W2 = np.zeros((3, 6), np.float32)
    for o, f in enumerate(feats):
        W1[2 * o, f], W1[2 * o + 1, f] = 1, -1
        W2[o, 2 * o], W2[o, 2 * o + 1] = 1, -1
    return oracle.Mlp([W1, W2], [np.zeros(6, np.float32), np.zeros(3, np.float32)], oracle.ACT_RELU)


def test_vhs_nn_features_read_back_through_a_probe_network():
    """With the energy shell off, g' = sigma_v * f(x); a pass-through network exposes x itself:
    x = [g/sigma_v (3), |g|/sigma_v, T_cell/T_scale, sigma_xi*xi (3)]  (eq. 1-3, Q1-Q3)."""
    pop = wl.couette(seed=3, n_cells=6, per_cell=400)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    prm = oracle.VhsParams(flags=oracle.F_NOISE, sigma_v=300.0, T_scale=250.0, noise_sigma=0.1)
    seg = lambda k: slice(cs[k], cs[k + 1])
    # features 0..2
    r = oracle.collide_vhs_nn(cs, *v, _probe_net(8, [0, 1, 2]), prm, 5, 2)
    ok = r.pair_i >= 0
    for k in range(pop.n_cells):
        base = cs[k]
        idx = np.flatnonzero(ok[seg(k)]) + base
        g = np.stack([a[base + r.pair_i[idx]] - a[base + r.pair_j[idx]] for a in v], axis=1)
        np.testing.assert_allclose(r.gprime[idx], g, rtol=1e-12, atol=1e-9)  # sigma_v * (g/sigma_v)
    # features 3, 4 (+ feature 5 = noise)
    r = oracle.collide_vhs_nn(cs, *v, _probe_net(8, [3, 4, 5]), prm, 5, 2)
    noise = []
    for k in range(pop.n_cells):
        base = cs[k]
        idx = np.flatnonzero(ok[seg(k)]) + base
        g = np.stack([a[base + r.pair_i[idx]] - a[base + r.pair_j[idx]] for a in v], axis=1)
        np.testing.assert_allclose(r.gprime[idx, 0], np.linalg.norm(g, axis=1), rtol=1e-12)
        Tk = M * sum(np.var(a[seg(k)]) for a in v) / (3 * KB)
        np.testing.assert_allclose(r.gprime[idx, 1], prm.sigma_v * Tk / prm.T_scale, rtol=1e-11)
        noise.append(r.gprime[idx, 2] / prm.sigma_v / prm.noise_sigma)
    noise = np.concatenate(noise)
    assert stats.kstest(noise, "norm").pvalue > 1e-3
    # noise flag off => the noise inputs are exactly zero
    prm.flags = 0
    r = oracle.collide_vhs_nn(cs, *v, _probe_net(8, [5, 6, 7]), prm, 5, 2)
    assert np.all(r.gprime[ok] == 0.0)
    # paper's 6-input form (Q1): (g/sigma_v) (+) xi
    prm.flags = oracle.F_NOISE
    r6 = oracle.collide_vhs_nn(cs, *v, _probe_net(6, [0, 1, 3]), prm, 5, 2)
    np.testing.assert_allclose(r6.gprime[ok, 2] / prm.sigma_v / prm.noise_sigma, noise, rtol=1e-9)


# ------------------------------------------------------------------------------------ P2/P3/P4
def _tiny_case(seed=0, n_cells=16, per_cell=100, H=32):
    pop = wl.tiny_box(seed=seed, n_cells=n_cells, per_cell=per_cell)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    Ws, bs = wl.random_mlp(seed, [8, H, H, 3])
    return cs, v, oracle.Mlp(Ws, bs, oracle.ACT_TANH)


def test_p2_pair_momentum_and_energy_are_conserved():
    """'guarantees conservation of pair momentum and (through (5)) pair kinetic energy'."""
    cs, v, net = _tiny_case()
    prm = oracle.VhsParams(flags=oracle.F_NOISE | oracle.F_ENERGY_SHELL, pairs_per_cell=50, sigma_v=wl.SIGMA_V)
    r = oracle.collide_vhs_nn(cs, *v, net, prm, 0, 0)
    new = [r.vx, r.vy, r.vz]
    n_pairs = 0
    for k in range(len(cs) - 1):
        for s in range(50):
            i, j = cs[k] + r.pair_i[cs[k] + s], cs[k] + r.pair_j[cs[k] + s]
            assert i != j
            for a in range(3):
                assert abs((new[a][i] + new[a][j]) - (v[a][i] + v[a][j])) <= 1e-13 * 1000
            e0 = sum(v[a][i] ** 2 + v[a][j] ** 2 for a in range(3))
            e1 = sum(new[a][i] ** 2 + new[a][j] ** 2 for a in range(3))
            assert abs(e1 - e0) <= 1e-13 * e0
            n_pairs += 1
    assert n_pairs == 16 * 50
    # disjointness: every slot appears at most once per cell
    for k in range(len(cs) - 1):
        used = np.concatenate([r.pair_i[cs[k]:cs[k] + 50], r.pair_j[cs[k]:cs[k] + 50]])
        assert len(np.unique(used)) == 100
    # unpaired particles untouched (pairs_per_cell = 50 of 100 uses everyone; use 10 here)
    prm.pairs_per_cell = 10
    r = oracle.collide_vhs_nn(cs, *v, net, prm, 0, 0)
    changed = (r.vx != v[0]) | (r.vy != v[1]) | (r.vz != v[2])
    assert changed.sum() <= 16 * 20


@pytest.mark.parametrize("shell", [True, False])
def test_p3_cell_moments_restored_by_matching(shell):
    """P:L134 'clamps the cell energy back to E_pre up to round-off'; P:L46 momentum and energy."""
    pop = wl.couette(seed=1, n_cells=8, per_cell=200)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    Ws, bs = wl.random_mlp(1, [8, 32, 32, 3])
    flags = oracle.F_NOISE | oracle.F_MOMENT_MATCH | (oracle.F_ENERGY_SHELL if shell else 0)
    prm = oracle.VhsParams(flags=flags, sigma_v=wl.SIGMA_V)
    pre = oracle.cell_moments(cs, *v)
    r = oracle.collide_vhs_nn(cs, *v, oracle.Mlp(Ws, bs), prm, 1, 0)
    post = oracle.cell_moments(cs, r.vx, r.vy, r.vz)
    N = np.diff(cs)
    scale = N * np.sqrt(pre[:, 3] / N)
    assert np.abs(post[:, :3] - pre[:, :3]).max() / scale.min() < 1e-12
    np.testing.assert_allclose(post[:, 3], pre[:, 3], rtol=1e-12)
    if not shell:  # without matching the same step does NOT conserve energy (negative control)
        prm.flags = oracle.F_NOISE
        r = oracle.collide_vhs_nn(cs, *v, oracle.Mlp(Ws, bs), prm, 1, 0)
        post = oracle.cell_moments(cs, r.vx, r.vy, r.vz)
        assert np.abs(post[:, 3] / pre[:, 3] - 1).max() > 1e-3


def test_p3_literal_eq11_restores_energy_only():
    pop = wl.couette(seed=2, n_cells=4, per_cell=100)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    Ws, bs = wl.random_mlp(1, [8, 16, 16, 3])
    prm = oracle.VhsParams(flags=oracle.F_NOISE | oracle.F_MOMENT_MATCH | oracle.F_MATCH_ENERGY_ONLY, sigma_v=wl.SIGMA_V)
    pre = oracle.cell_moments(cs, *v)
    r = oracle.collide_vhs_nn(cs, *v, oracle.Mlp(Ws, bs), prm, 1, 0)
    post = oracle.cell_moments(cs, r.vx, r.vy, r.vz)
    np.testing.assert_allclose(post[:, 3], pre[:, 3], rtol=1e-12)
    assert np.abs(post[:, 0] - pre[:, 0]).max() > 1e-6  # momentum is NOT restored by eq. 11 alone


def test_p4_no_artificial_cooling_over_100_steps():
    """noise + rescaling keeps T; shell off + matching off cools."""
    cs, v, net = _tiny_case(seed=0, n_cells=8, per_cell=100, H=16)
    prm = oracle.VhsParams(pairs_per_cell=50, sigma_v=wl.SIGMA_V)
    T0 = np.array([oracle.cell_state(*[a[cs[k]:cs[k + 1]] for a in v], M)[2] for k in range(8)])
    cur = v
    for t in range(100):
        r = oracle.collide_vhs_nn(cs, *cur, net, prm, 0, t)
        cur = [r.vx, r.vy, r.vz]
    T1 = np.array([oracle.cell_state(*[a[cs[k]:cs[k + 1]] for a in cur], M)[2] for k in range(8)])
    np.testing.assert_allclose(T1, T0, rtol=1e-12)
    assert np.abs(cur[0] - v[0]).max() > 1.0  # the gas did evolve
    prm.flags = oracle.F_NOISE  # negative control
    cur = v
    for t in range(10):
        r = oracle.collide_vhs_nn(cs, *cur, net, prm, 0, t)
        cur = [r.vx, r.vy, r.vz]
    T2 = np.array([oracle.cell_state(*[a[cs[k]:cs[k + 1]] for a in cur], M)[2] for k in range(8)])
    assert np.all(np.abs(T2 / T0 - 1) > 0.05)


def test_p10_moment_match_algebra_and_identity():
    rng = np.random.default_rng(3)
    cs = np.array([0, 50, 51, 51, 200], np.int32)
    v = rng.normal(50, 200, (3, 200))
    tgt = oracle.cell_moments(cs, *rng.normal(-20, 150, (3, 200)))
    out = oracle.moment_match(cs, *v, tgt)
    got = oracle.cell_moments(cs, *out)
    for k in (0, 3):
        np.testing.assert_allclose(got[k], tgt[k], rtol=1e-12, atol=1e-9)
    for a in range(3):  # N<2 cells untouched (Q11)
        np.testing.assert_array_equal(out[a][50:51], v[a][50:51])
    same = oracle.moment_match(cs, *v, oracle.cell_moments(cs, *v))
    for a in range(3):
        np.testing.assert_allclose(same[a], v[a], rtol=1e-13, atol=1e-11)


# ------------------------------------------------------------------------------------ P5 VHS rate
def test_p5_vhs_collision_rate_closed_form():
    """<sigma_T c_r>_Maxwell(T) = 4 d_ref^2 sqrt(pi kB T_ref/m) (T/T_ref)^(1-omega) (Bird's VHS rate)."""
    prm = oracle.VhsParams()
    for T in (200.0, 273.0, 1000.0, 7000.0):
        a = M / (4 * KB * T)  # relative-speed pdf: 4 pi (a/pi)^1.5 g^2 exp(-a g^2), m_r = m/2
        pdf = lambda g: 4 * math.pi * (a / math.pi) ** 1.5 * g * g * math.exp(-a * g * g)
        gs = math.sqrt(1 / a)
        num, _ = integrate.quad(lambda g: oracle.vhs_sigma_g(g, prm) * pdf(g), 0, 12 * gs, epsabs=0, epsrel=1e-11, limit=200)
        closed = 4 * prm.d_ref ** 2 * math.sqrt(math.pi * KB * prm.T_ref / M) * (T / prm.T_ref) ** (1 - prm.omega)
        assert abs(num / closed - 1) < 1e-8


def test_p5_acceptance_fraction_matches_rate_ratio():
    pop = wl.tiny_box(seed=9, n_cells=40, per_cell=1000)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    prm = oracle.VhsParams(flags=oracle.F_ACCEPT | oracle.F_ENERGY_SHELL | oracle.F_NOISE, sigma_v=wl.SIGMA_V)
    cap = oracle.vhs_sigma_g(6 * wl.SIGMA_V, prm)
    Ws, bs = wl.random_mlp(0, [8, 8, 8, 3])
    r = oracle.collide_vhs_nn(cs, *v, oracle.Mlp(Ws, bs), prm, 4, 0, sigma_cr_max=np.full(40, cap, np.float32))
    ok = r.pair_i >= 0
    frac = r.accepted[ok].mean()
    closed = 4 * prm.d_ref ** 2 * math.sqrt(math.pi * KB * prm.T_ref / M) / float(np.float32(cap))
    n = ok.sum()
    assert n == 20000 and abs(frac - closed) < 4 * math.sqrt(closed * (1 - closed) / n)
    # rejected pairs keep their velocities
    rej = np.flatnonzero(ok & (r.accepted == 0))
    k = np.searchsorted(cs, rej, side="right") - 1
    i = cs[k] + r.pair_i[rej]
    assert np.all(r.vx[i] == v[0][i])


# ------------------------------------------------------------------------------------ P13 rotation
def test_p13_rotation_invariants_and_special_cases():
    rng = np.random.default_rng(5)
    for _ in range(200):
        g = rng.normal(0, 500, 3)
        chi, eps = rng.uniform(0, 2 * math.pi, 2)
        gp = oracle.rotate(g, chi, eps)
        assert abs(np.linalg.norm(gp) / np.linalg.norm(g) - 1) < 1e-14
        assert abs(np.dot(g, gp) / np.dot(g, g) - math.cos(chi)) < 1e-14
    np.testing.assert_allclose(oracle.rotate([3.0, 0, 0], math.pi / 2, 0.0), [0, 3, 0], atol=1e-15)
    np.testing.assert_allclose(oracle.rotate([-3.0, 0, 0], math.pi / 2, math.pi / 2), [0, 0, 3], atol=1e-15)
    np.testing.assert_allclose(oracle.rotate([0, 2.0, 0], math.pi / 2, math.pi / 2), [2, 0, 0], atol=1e-15)
    np.testing.assert_allclose(oracle.rotate([1.0, 2.0, 3.0], 0.0, 1.234), [1, 2, 3], atol=1e-15)
    np.testing.assert_allclose(oracle.rotate([1.0, 2.0, 3.0], math.pi, 0.3), [-1, -2, -3], atol=1e-14)
    # hard-sphere sampling (cos chi uniform, eps uniform) must give an isotropic g'
    U = rng.random((20000, 2))
    gp = np.array([oracle.rotate([1.0, 2.0, -0.5], 2 * math.acos(math.sqrt(u[0])), 2 * math.pi * u[1]) for u in U])
    gp /= math.sqrt(5.25)
    assert np.abs(gp.mean(axis=0)).max() < 4 / math.sqrt(3 * 20000)
    assert np.abs((gp ** 2).mean(axis=0) - 1 / 3).max() < 0.01


# ------------------------------------------------------------------------------------ P6/P7/P8 chi
def test_p6_hard_sphere_deflection():
    hs = oracle.Potential(oracle.POT_HARD_SPHERE, 4.17e-10, 0.0, 5 * 4.17e-10)
    for bd in (0.0, 0.1, 0.5, 0.9, 0.999):
        chi = oracle.chi_exact(hs, 300 * KB, bd * 4.17e-10, 8)
        assert abs(chi - 2 * math.acos(bd)) < 1e-12
    assert abs(oracle.chi_exact(hs, 300 * KB, 1.5 * 4.17e-10, 8)) < 1e-10  # miss


def test_p7_coulomb_and_inverse_square_closed_forms():
    for kappa, E, b in ((1.0, 1.0, 0.5), (1.0, 0.2, 2.0), (3.0, 5.0, 0.1), (-0.3, 1.0, 1.0)):
        pot = oracle.Potential(oracle.POT_INV_R, kappa, 0.0, 100.0)
        ref = 2 * math.atan(kappa / (2 * E * b))  # Rutherford
        assert abs(oracle.chi_exact(pot, E, b, 32) - ref) < 2e-9
    for kappa, E, b in ((1.0, 1.0, 0.5), (2.0, 0.5, 1.5), (0.1, 3.0, 0.05)):
        pot = oracle.Potential(oracle.POT_INV_R2, kappa, 0.0, 100.0)
        ref = math.pi * (1 - b / math.sqrt(b * b + kappa / E))
        assert abs(oracle.chi_exact(pot, E, b, 32) - ref) < 2e-9


def _chi_scipy(E, b):
    """The paper's own recipe on LJ in reduced units: brentq for the largest root,
    u = r_min/r substitution, scipy quad with the algebraic end-point weight."""
    V = lambda r: 4 * (r ** -12 - r ** -6)
    F = lambda r: 1 - b * b / (r * r) - V(r) / E
    rs = np.geomspace(50.0, 0.3, 20000)
    Fs = F(rs)
    idx = np.argmax(Fs < 0)
    rmin = optimize.brentq(F, rs[idx], rs[idx - 1], xtol=1e-15, rtol=1e-15)
    beta = b / rmin
    Ft = lambda u: 1 - beta * beta * u * u - V(rmin / u) / E if u > 0 else 1.0
    # integrand = h(u) (1-u)^(-1/2) with h smooth: quad's 'alg' weight handles the end point
    h = lambda u: math.sqrt((1 - u) / max(Ft(u), 1e-300)) if u < 1 else 0.0
    val, _ = integrate.quad(h, 0, 1, weight="alg", wvar=(0, -0.5), epsabs=1e-13, epsrel=1e-12, limit=400)
    return math.pi - 2 * beta * val


def test_p8_lj_worked_values_and_scipy_recipe():
    lj = oracle.Potential(oracle.POT_LJ, 1.0, 1.0, 10.0)
    for line in open(os.path.join(GOLD, "lj_chi_worked_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        E, b, ref = map(float, line.split())
        got = oracle.chi_exact(lj, E, b, 4)
        assert abs(got - ref) < 1e-9
        assert abs(got - _chi_scipy(E, b)) < 5e-8
        assert abs(oracle.chi_exact(lj, E, b, 16) - got) < 1e-9  # quadrature converged


def test_lj_argon_units_and_rmin_root():
    lj = oracle.lj_argon()
    # reduced-unit invariance: chi depends only on E/eps and b/sigma
    ref = oracle.chi_exact(oracle.Potential(oracle.POT_LJ, 1.0, 1.0, 10.0), 58.43, 0.5, 4)
    assert abs(oracle.chi_exact(lj, 58.43 * 119.8 * KB, 0.5 * 3.405e-10, 4) - ref) < 1e-10
    E, b = 2.0 * 119.8 * KB, 1.2 * 3.405e-10
    r = oracle.rmin(lj, E, b)
    F = 1 - b * b / (r * r) - oracle.potential_eval(lj, r) / E
    assert 0 <= F < 1e-12
    assert abs(oracle.potential_eval(lj, 3.405e-10)) < 1e-30 * 1e9  # V(sigma) = 0
    assert abs(oracle.potential_eval(lj, 2 ** (1 / 6) * 3.405e-10) / (119.8 * KB) + 1) < 1e-12  # well depth


# ------------------------------------------------------------------------------------ P9 table
def test_p9_bilinear_is_exact_on_bilinear_functions_and_clamps():
    nE, nB = 9, 7
    lo, hi = math.log(5.0), math.log(6e4)
    Eg = lo + (hi - lo) * np.arange(nE) / (nE - 1)
    Bg = np.arange(nB) / (nB - 1)
    f = lambda e, b: 0.5 + 0.25 * e - 1.5 * b + 0.125 * e * b
    tab = oracle.ChiTable(f(Eg[:, None], Bg[None, :]).astype(np.float64).astype(np.float32), lo, hi)
    exact = lambda e, b: float(np.float32(1.0)) * f(e, b)
    rng = np.random.default_rng(0)
    for _ in range(200):
        e, b = rng.uniform(lo, hi), rng.random()
        assert abs(oracle.chi_bilinear(tab, e, b) - exact(e, b)) < 2e-6  # fp32 node rounding only
    assert abs(oracle.chi_bilinear(tab, lo - 5, 0.3) - exact(lo, 0.3)) < 2e-6
    assert abs(oracle.chi_bilinear(tab, hi + 5, 1.7) - exact(hi, 1.0)) < 2e-6
    assert abs(oracle.chi_bilinear(tab, -math.inf, -0.1) - exact(lo, 0.0)) < 2e-6
    # node values are returned exactly, E-major layout chi[iE*nB+iB]
    assert oracle.chi_bilinear(tab, Eg[3], Bg[5]) == pytest.approx(float(tab.chi[3, 5]), abs=1e-6)


def test_table_built_from_quadrature_and_interpolation_error():
    lj = oracle.lj_argon()
    tab = oracle.build_chi_table(lj, 33, 33, n_panels=2)
    lo, hi = tab.lnE_min, tab.lnE_max
    assert tab.chi[:, 0] == pytest.approx(math.pi, abs=1e-6)  # head-on
    for iE, iB in ((5, 7), (20, 3), (32, 32), (12, 30)):
        E = KB * math.exp(lo + (hi - lo) * iE / 32)
        assert tab.chi[iE, iB] == pytest.approx(abs(oracle.chi_exact(lj, E, 1e-9 * iB / 32, 8)), abs=1e-6)
    assert np.all(tab.chi >= 0)  # Q14: |chi|


def test_chi_mlp_head_is_exp_and_inputs_are_normalised():
    """softplus output trained on ln(1+chi): chi = expm1(softplus(z)) = e^z."""
    lo, hi = math.log(5.0), math.log(6e4)
    W1 = np.array([[1, 0], [0, 1]], np.float32)
    net = oracle.Mlp([W1, np.array([[2.0, -3.0]], np.float32)], [np.zeros(2, np.float32), np.array([0.25], np.float32)], oracle.ACT_RELU)
    for lnE, bt in ((3.0, 0.2), (9.5, 0.9), (lo, 0.0), (hi, 1.0)):
        x0 = (lnE - lo) / (hi - lo)
        assert oracle.chi_mlp(net, lo, hi, lnE, bt) == pytest.approx(math.exp(2 * x0 - 3 * bt + 0.25), rel=1e-12)
    assert oracle.chi_mlp(net, lo, hi, lo - 3, 1.5) == pytest.approx(math.exp(-3 + 0.25), rel=1e-12)  # clamps
    assert oracle.chi_mlp(net, lo, hi, hi + 3, -1.0) == pytest.approx(math.exp(2 + 0.25), rel=1e-12)


def test_abinitio_step_plumbing_via_probe_tables():
    """Tables that return b~ or E~ expose what the step feeds the lookup: b~ = sqrt(U_b),
    E~ = ln(m g^2 / (4 kB))  (P:L334 with mu = m/2)."""
    pop = wl.tiny_box(seed=11, n_cells=10, per_cell=400, T=1000.0)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    lo, hi = math.log(5.0), math.log(6e4)
    nE = nB = 17
    tb = oracle.ChiTable(np.tile(np.arange(nB) / (nB - 1), (nE, 1)).astype(np.float32), lo, hi)
    prm = oracle.AbinitioParams(flags=0)
    r = oracle.collide_abinitio(cs, *v, prm, 21, 3, table=tb)
    ok = r.pair_i >= 0
    assert ok.sum() == 2000
    assert stats.kstest(r.aux[ok] ** 2, "uniform").pvalue > 1e-3  # chi = b~ = sqrt(U) => chi^2 ~ U(0,1)
    te = oracle.ChiTable(np.tile((lo + (hi - lo) * np.arange(nE) / (nE - 1))[:, None], (1, nB)).astype(np.float32), lo, hi)
    r = oracle.collide_abinitio(cs, *v, prm, 21, 3, table=te)
    idx = np.flatnonzero(ok)
    k = np.searchsorted(cs, idx, side="right") - 1
    g2 = sum((a[cs[k] + r.pair_i[idx]] - a[cs[k] + r.pair_j[idx]]) ** 2 for a in v)
    lnE = np.clip(np.log(M * g2 / (4 * KB)), lo, hi)
    np.testing.assert_allclose(r.aux[idx], lnE, atol=2e-6)
    # rotation really uses chi: |g'| = |g| and cos angle = cos chi; pair invariants hold
    gp = r.gprime[idx]
    g = np.stack([a[cs[k] + r.pair_i[idx]] - a[cs[k] + r.pair_j[idx]] for a in v], axis=1)
    np.testing.assert_allclose(np.linalg.norm(gp, axis=1), np.sqrt(g2), rtol=1e-13)
    np.testing.assert_allclose((g * gp).sum(axis=1) / g2, np.cos(r.aux[idx]), atol=1e-13)
    pre, post = oracle.cell_moments(cs, *v), oracle.cell_moments(cs, r.vx, r.vy, r.vz)
    np.testing.assert_allclose(post[:, 3], pre[:, 3], rtol=1e-13)
    np.testing.assert_allclose(post[:, :3], pre[:, :3], atol=1e-8)
    # azimuth: eps = 2 pi U_eps uniform => with chi = pi/2 the component of g' along any fixed
    # direction perpendicular to g averages to zero
    th = oracle.ChiTable(np.full((nE, nB), math.pi / 2, np.float32), lo, hi)
    r = oracle.collide_abinitio(cs, *v, prm, 21, 3, table=th)
    gp = r.gprime[idx] / np.sqrt(g2)[:, None]
    assert np.abs(gp.mean(axis=0)).max() < 4.5 / math.sqrt(3 * len(idx))


def test_abinitio_acceptance_constant_cross_section():
    pop = wl.tiny_box(seed=12, n_cells=20, per_cell=1000, T=500.0)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    tb = oracle.ChiTable(np.full((4, 4), 1.0, np.float32), math.log(5.0), math.log(6e4))
    gmax = 6 * math.sqrt(2 * KB * 500.0 / M)
    prm = oracle.AbinitioParams(flags=oracle.F_ACCEPT)
    r = oracle.collide_abinitio(cs, *v, prm, 2, 0, table=tb, cr_max=np.full(20, gmax, np.float32))
    ok = r.pair_i >= 0
    mean_g = math.sqrt(16 * KB * 500.0 / (math.pi * M))  # <g> = sqrt(8 kB T/(pi m_r))
    p = mean_g / float(np.float32(gmax))
    assert abs(r.accepted[ok].mean() - p) < 4 * math.sqrt(p * (1 - p) / ok.sum())


def test_chi_batch_matches_pointwise_calls():
    lj = oracle.lj_argon()
    tab = oracle.build_chi_table(lj, 17, 17, n_panels=2)
    E, b = wl.abinitio_pair_batch(seed=3, n=500)
    out = oracle.chi_batch(E, b, 0, 1e-9, table=tab)
    for p in (0, 17, 499):
        assert out[p] == oracle.chi_bilinear(tab, math.log(float(E[p])), float(b[p]) / 1e-9)
    Ws, bs = wl.random_mlp(3, [2, 16, 16, 1])
    net = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    out = oracle.chi_batch(E, b, 1, 1e-9, net=net)
    assert out[5] == oracle.chi_mlp(net, math.log(5.0), math.log(6e4), math.log(float(E[5])), float(b[5]) / 1e-9)
    assert np.all(out > 0)


def test_workload_shapes_match_baseline_configs():
    assert wl.tiny_box().n == 6400
    p = wl.mach10_cylinder(nx=40, ny=20, n_total=200000)
    assert p.n == 200000 and (p.counts == 0).sum() > 0
    ratio = np.sort(np.unique(p.counts[p.counts > 0]))
    assert ratio[-1] / ratio[0] > 15  # 16x density contrast between shock band and wake
    rc, perm, cs = oracle.bin_particles(p.cell, p.n_cells)
    np.testing.assert_array_equal(np.diff(cs), p.counts)


def test_chapman_enskog_collision_integral_of_lj_matches_textbook():
    """Pin P14 (physics level, independent of the oracle): the deflection angles of the oracle's quadrature,
    pushed through Q^(2)(E) = 2 pi int (1 - cos^2 chi) b db (eq. 19) and the Maxwellian average of eq. 18
    in its standard Chapman-Enskog form, must reproduce the tabulated reduced collision integral Omega^(2,2)* of
    the Lennard-Jones gas (tests/golden/lj_omega22_textbook.txt).  A wrong sign, a wrong root or a dropped factor
    in the quadrature moves these numbers by far more than the 0.5 % allowed here."""
    pot = oracle.lj_argon()
    eps, sig = 119.8 * KB, 3.405e-10
    rows = [l.split() for l in open(os.path.join(GOLD, "lj_omega22_textbook.txt")) if l.strip() and not l.startswith("#")]
    xs, ws = np.polynomial.laguerre.laggauss(20)
    nb, bmax = 400, 4.0
    bs = (np.arange(nb) + 0.5) * bmax / nb

    def q2_star(Es):
        chi = np.array([oracle.chi_exact(pot, Es * eps, b * sig) for b in bs])
        return 3.0 * np.sum((1.0 - np.cos(chi) ** 2) * bs) * bmax / nb

    for Ts, want in ((float(r[0]), float(r[1])) for r in rows):
        got = sum(w * x ** 3 * q2_star(x * Ts) for x, w in zip(xs, ws)) / 6.0
        assert abs(got / want - 1.0) < 5e-3, (Ts, got, want)


def test_with_replacement_selection_and_batch_semantics():
    """NTC-style selection WITH replacement ("two particles i, j in C_k are selected uniformly
    at random") and batch evaluation.  Pins: (a) the draw is uniform over ORDERED pairs i != j (brute
    force, N = 3, 4, 7); (b) a brute-force re-computation of one cell from the dumped pairs: every pair is evaluated
    on the PRE-collision velocities and the changes add up; (c) momentum is conserved exactly before matching while
    energy is not; (d) matching restores both."""
    for N in (3, 4, 7):
        n = 3000 * N * (N - 1)
        cnt = {}
        for s in range(n):
            ij = oracle.pair_draw(77, 5, 9, s, N)
            assert ij[0] != ij[1] and 0 <= ij[0] < N and 0 <= ij[1] < N
            cnt[ij] = cnt.get(ij, 0) + 1
        assert len(cnt) == N * (N - 1)
        p = 1.0 / (N * (N - 1))
        for c in cnt.values():
            assert abs(c / n - p) < 4.5 * math.sqrt(p * (1 - p) / n)
    # the draw is what its definition says: mulhi of the first two words of stream 4
    r = oracle.philox4x32_10([11, 9, 5, 4], [77, 0])
    i = (r[0] * 7) >> 32
    j = (r[1] * 6) >> 32
    assert oracle.pair_draw(77, 5, 9, 11, 7) == (i, j + (1 if j >= i else 0))

    pop = wl.tiny_box(seed=13, n_cells=6, per_cell=40, T=800.0)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    lo, hi = math.log(5.0), math.log(6e4)
    tb = oracle.ChiTable(np.full((4, 4), 1.3, np.float32), lo, hi)  # chi = 1.3 rad for every pair
    prm = oracle.AbinitioParams(flags=oracle.F_PAIR_REPLACE)      # no matching
    r = oracle.collide_abinitio(cs, *v, prm, 31, 2, table=tb)
    ok = r.pair_i >= 0
    assert ok.sum() == 6 * 20
    # (b) brute force for every cell from the dumped (i, j, g')
    for k in range(pop.n_cells):
        a, N = cs[k], cs[k + 1] - cs[k]
        loc = np.stack([x[a:a + N] for x in v], axis=1)
        dv = np.zeros_like(loc)
        for s in range(N // 2):
            i, j = r.pair_i[a + s], r.pair_j[a + s]
            assert (i, j) == oracle.pair_draw(31, 2, k, s, N)
            g = loc[i] - loc[j]
            gp = r.gprime[a + s]
            assert abs(np.linalg.norm(gp) / np.linalg.norm(g) - 1) < 1e-13          # rotation keeps |g|
            assert abs(np.dot(g, gp) / np.dot(g, g) - math.cos(1.3)) < 1e-6         # by chi (fp32 table value)
            dv[i] += 0.5 * (gp - g)
            dv[j] -= 0.5 * (gp - g)
        got = np.stack([r.vx[a:a + N], r.vy[a:a + N], r.vz[a:a + N]], axis=1)
        np.testing.assert_allclose(got, loc + dv, rtol=0, atol=1e-9)
    # (c) momentum exact, energy not (a particle in several pairs takes all their changes)
    pre, post = oracle.cell_moments(cs, *v), oracle.cell_moments(cs, r.vx, r.vy, r.vz)
    np.testing.assert_allclose(post[:, :3], pre[:, :3], atol=1e-8)
    assert np.abs(post[:, 3] / pre[:, 3] - 1).max() > 1e-3
    # about a quarter of the particles appear in two or more pairs at M = N / 2
    multi = np.mean([np.bincount(np.r_[r.pair_i[cs[k]:cs[k] + 20], r.pair_j[cs[k]:cs[k] + 20]], minlength=40).max() >= 2
                     for k in range(6)])
    assert multi == 1.0
    # (d) with matching both are restored
    r2 = oracle.collide_abinitio(cs, *v, oracle.AbinitioParams(flags=oracle.F_PAIR_REPLACE | oracle.F_MOMENT_MATCH), 31, 2, table=tb)
    post2 = oracle.cell_moments(cs, r2.vx, r2.vy, r2.vz)
    np.testing.assert_allclose(post2[:, 3], pre[:, 3], rtol=1e-12)
    np.testing.assert_allclose(post2[:, :3], pre[:, :3], atol=1e-8)


# --------------------------------------------------------------- f1: NTC candidate count, carried remainder
def test_ntc_counts_formula_remainder_and_time_average():
    """count = floor(1/2 N (N-1) coef max + R) ("proportional to N_k (N_k - 1) and ... (sigma v_r)max,k"),
    the fraction is carried: over T steps the counts add up to floor(T m) and never differ from m by one or more."""
    cs = np.array([0, 10, 11, 11, 31, 131], np.int32)
    cap = np.array([1.0, 5.0, 7.0, 2.0, 0.37], np.float32)
    coef = 0.0123
    R = np.zeros(5)
    N = np.diff(cs).astype(np.float64)
    m = 0.5 * N * (N - 1) * coef * cap.astype(np.float64)
    total = np.zeros(5, np.int64)
    for t in range(1, 401):
        c = oracle.ntc_counts(cs, cap, coef, R)
        total += c
        assert np.all(c >= np.floor(m)) and np.all(c <= np.floor(m) + 1)
        assert np.all((R >= 0) & (R < 1))
        assert np.all(np.abs(total - t * m) < 1.0)          # the running total tracks t m to within one pair
    assert list(total[1:3]) == [0, 0]                       # N = 1 and N = 0: no candidates
    assert abs(R[0] - (400 * m[0] - total[0])) < 1e-9
    # a remainder handed in is honoured
    R = np.array([0.75, 0, 0, 0, 0])
    c = oracle.ntc_counts(cs, cap, coef, R)
    assert c[0] == math.floor(m[0] + 0.75) and abs(R[0] - (m[0] + 0.75 - c[0])) < 1e-12


def test_ntc_equilibrium_collision_frequency_closed_form():
    """NTC candidates x acceptance reproduce the equilibrium VHS collision rate (Bird 1994 eq. 4.64):
    accepted collisions per cell and step = 1/2 N (N-1) coef <sigma_T c_r>, <sigma_T c_r> = nu / n =
    4 d_ref^2 sqrt(pi kB T_ref / m) (T / T_ref)^(1 - omega); checked at T = 400 K so the exponent matters."""
    T = 400.0
    K, N, steps = 200, 200, 6
    pop = wl.tiny_box(seed=21, n_cells=K, per_cell=N, T=T)
    rc, perm, cs = oracle.bin_particles(pop.cell, K)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    base = oracle.VhsParams(flags=oracle.F_ACCEPT | oracle.F_ENERGY_SHELL | oracle.F_NOISE, sigma_v=wl.SIGMA_V)
    cap = np.full(K, oracle.vhs_sigma_g(8 * wl.SIGMA_V, base), np.float32)
    rate = 4 * base.d_ref ** 2 * math.sqrt(math.pi * KB * base.T_ref / M) * (T / base.T_ref) ** (1 - base.omega)
    coef = 24.3 / (0.5 * N * (N - 1) * float(cap[0]))       # 24.3 candidates per cell and step
    Ws, bs = wl.random_mlp(0, [8, 8, 8, 3])
    R = np.zeros(K)
    cand = acc = 0
    for t in range(steps):
        counts = oracle.ntc_counts(cs, cap, coef, R)
        prm = oracle.VhsParams(flags=base.flags, sigma_v=wl.SIGMA_V, pairs_count=counts)
        r = oracle.collide_vhs_nn(cs, *v, oracle.Mlp(Ws, bs), prm, 4, t, sigma_cr_max=cap)
        ok = r.pair_i >= 0
        assert ok.sum() == counts.sum()                      # every cell ran exactly its own count
        cand += ok.sum()
        acc += r.accepted[ok].sum()
        v = [r.vx, r.vy, r.vz]                               # energy-shell collisions keep the gas at T
    assert abs(cand - steps * K * 24.3) < K                  # carried remainders: within one pair per cell
    want = steps * K * 0.5 * N * (N - 1) * coef * rate
    assert abs(acc - want) < 4 * math.sqrt(want)             # Poisson scatter of the accepted count


def test_with_replacement_vhs_nn_batch_semantics():
    """SURVEY 8(f1) for the VHS-surrogate operator: the same with-replacement draw and batch semantics as the ab
    initio step.  Brute force from the dumped pairs: g' recomputed with the MLP evaluated by numpy on the
    PRE-collision relative velocity (features of Q2/Q3, energy-shell projection eq. 5), changes added up; momentum
    exact, energy restored only by the matching."""
    pop = wl.tiny_box(seed=17, n_cells=5, per_cell=36, T=300.0)
    rc, perm, cs = oracle.bin_particles(pop.cell, pop.n_cells)
    v = [a[perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    Ws, bs = wl.random_mlp(6, [8, 16, 16, 3])
    net = oracle.Mlp(Ws, bs, oracle.ACT_TANH)
    flags = oracle.F_PAIR_REPLACE | oracle.F_ENERGY_SHELL          # no noise: the features are deterministic
    prm = oracle.VhsParams(sigma_v=wl.SIGMA_V, flags=flags)
    r = oracle.collide_vhs_nn(cs, *v, net, prm, 5, 3)
    assert (r.pair_i >= 0).sum() == 5 * 18
    for k in range(pop.n_cells):
        a, N = cs[k], cs[k + 1] - cs[k]
        loc = np.stack([x[a:a + N] for x in v], axis=1)
        ubar = loc.mean(axis=0)
        Tk = M * ((loc - ubar) ** 2).sum() / (3 * KB * N)           # eq. 10 cell temperature (Q3)
        dv = np.zeros_like(loc)
        for s in range(N // 2):
            i, j = r.pair_i[a + s], r.pair_j[a + s]
            assert (i, j) == oracle.pair_draw(5, 3, k, s, N)
            g = loc[i] - loc[j]
            gn = np.linalg.norm(g)
            h = np.concatenate([g / wl.SIGMA_V, [gn / wl.SIGMA_V, Tk / 273.0, 0.0, 0.0, 0.0]])
            for l, (W, b) in enumerate(zip(Ws, bs)):
                h = W.astype(np.float64) @ h + b.astype(np.float64)
                if l < len(Ws) - 1:
                    h = np.tanh(h)
            gp = gn * h / np.linalg.norm(h)
            np.testing.assert_allclose(r.gprime[a + s], gp, rtol=1e-10, atol=1e-9)
            dv[i] += 0.5 * (gp - g)
            dv[j] -= 0.5 * (gp - g)
        got = np.stack([r.vx[a:a + N], r.vy[a:a + N], r.vz[a:a + N]], axis=1)
        np.testing.assert_allclose(got, loc + dv, rtol=0, atol=1e-9)
    pre, post = oracle.cell_moments(cs, *v), oracle.cell_moments(cs, r.vx, r.vy, r.vz)
    np.testing.assert_allclose(post[:, :3], pre[:, :3], atol=1e-8)
    assert np.abs(post[:, 3] / pre[:, 3] - 1).max() > 1e-3
    r2 = oracle.collide_vhs_nn(cs, *v, net, oracle.VhsParams(sigma_v=wl.SIGMA_V, flags=flags | oracle.F_MOMENT_MATCH), 5, 3)
    post2 = oracle.cell_moments(cs, r2.vx, r2.vy, r2.vz)
    np.testing.assert_allclose(post2[:, 3], pre[:, 3], rtol=1e-12)
    np.testing.assert_allclose(post2[:, :3], pre[:, :3], atol=1e-8)


def test_table_builder_caps_non_finite_nodes_at_64_pi():
    """Q23: a node on the orbiting singularity has no finite deflection angle; the table builder stores 64 pi (32
    revolutions) there and leaves every smaller angle alone.  The quadrature itself never returns a non-finite value on
    the grids used here, so the cap is pinned at its own seam (the function orc_build_chi_table applies to every node):
    +inf, NaN and anything above 64 pi give 64 pi exactly, everything else passes unchanged; and a real LJ table stays
    far below the cap."""
    cap = 64.0 * np.pi
    assert oracle.cap_chi(float("inf")) == cap
    assert oracle.cap_chi(float("nan")) == cap  # a comparison written as c > cap would let NaN through
    assert oracle.cap_chi(cap * 1.0000001) == cap and oracle.cap_chi(1e300) == cap
    for c in (0.0, 1e-12, np.pi, 17.25, cap):
        assert oracle.cap_chi(c) == c
    assert np.isfinite(np.float32(cap))
    good = oracle.build_chi_table(oracle.lj_argon(), 8, 9, n_panels=1)
    assert np.all(np.isfinite(good.chi)) and good.chi.max() < 4 * np.pi and np.all(good.chi >= 0)


def test_neural_table_builder_nodes_closed_form_and_lookup():
    """f2, orc_build_chi_table_mlp: with a linear probe network the head makes chi = exp(z) (expm1 o softplus),
    so node (i, j) must hold exp(a i/(nE-1) + c j/(nB-1) + d) to fp32 rounding: pins the node coordinates of Q13
    (row = energy, column = impact parameter, both ends included) and the abs / cap seam; a lookup through the table
    at the nodes returns the node; a real SiLU network's table equals orc_chi_mlp at the node coordinates."""
    a, c, d = 1.75, -2.5, 0.25  # exact in fp32
    net = oracle.Mlp([np.array([[a, c]], np.float32)], [np.array([d], np.float32)], oracle.ACT_SILU)
    lo, hi = math.log(5.0), math.log(6e4)
    nE, nB = 7, 5
    tab = oracle.build_chi_table_mlp(net, nE, nB, lo, hi)
    assert tab.chi.shape == (nE, nB) and tab.chi.dtype == np.float32
    i, j = np.meshgrid(np.arange(nE), np.arange(nB), indexing="ij")
    want = np.exp(a * i / (nE - 1) + c * j / (nB - 1) + d)
    np.testing.assert_allclose(tab.chi, want, rtol=6e-8)  # half an fp32 ulp: the rounding of the stored node
    assert tab.chi[nE - 1, 0] == pytest.approx(math.exp(a + d), rel=6e-8) and tab.chi[0, nB - 1] == pytest.approx(math.exp(c + d), rel=6e-8)
    for ii, jj in ((0, 0), (3, 2), (nE - 1, nB - 1), (5, 1)):
        got = oracle.chi_bilinear(tab, lo + (hi - lo) * ii / (nE - 1), jj / (nB - 1))
        assert got == pytest.approx(float(tab.chi[ii, jj]), rel=1e-12)
    # a network whose output would exceed the cap: exp(6) = 403 > 64 pi = 201 -> capped (Q23)
    big = oracle.Mlp([np.array([[0.0, 0.0]], np.float32)], [np.array([6.0], np.float32)], oracle.ACT_SILU)
    assert np.all(oracle.build_chi_table_mlp(big, 3, 3, lo, hi).chi == np.float32(64 * np.pi))
    # hidden layers: the table is orc_chi_mlp at the node coordinates
    rng = np.random.default_rng(5)
    Ws = [rng.uniform(-1, 1, (16, 2)).astype(np.float32), rng.uniform(-0.3, 0.3, (1, 16)).astype(np.float32)]
    bs = [rng.uniform(-1, 1, 16).astype(np.float32), np.array([0.1], np.float32)]
    deep = oracle.Mlp(Ws, bs, oracle.ACT_SILU)
    t2 = oracle.build_chi_table_mlp(deep, 4, 6, lo, hi)
    for ii, jj in ((0, 0), (1, 4), (3, 5), (2, 2)):
        assert t2.chi[ii, jj] == np.float32(oracle.chi_mlp(deep, lo, hi, lo + (hi - lo) * ii / 3, jj / 5))

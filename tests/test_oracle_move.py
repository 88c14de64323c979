"""Pins for the oracle's minimal DSMC loop pieces, SURVEY.md 8(f4) (-m "not gpu"): free flight + Maxwell walls
for the 1-D Couette layout (reading Q30) and the per-cell sampling sums.  Each test checks the
oracle against something other than itself: the closed-form triangle-wave fold of specular reflection, the moments
of the flux-weighted wall Maxwellian, the textbook free-molecular Couette shear stress, brute-force sums."""
import math

import numpy as np

import oracle

RT = 208.13 * 273.0  # k_B T / m of argon at 273 K [m^2/s^2]


def _gas(n, seed, L=1.0, rt=RT):
    rng = np.random.default_rng(seed)
    return rng.random(n) * L, rng.normal(0.0, math.sqrt(rt), (3, n))


def test_specular_walls_fold_like_a_triangle_wave():
    """accommodation = 0: x(t) of a ball between two mirrors is the triangle wave of period 2L; |vx| is kept and
    its sign flips once per wall hit; vy, vz untouched; the random numbers play no role."""
    L, dt = 0.37, 1.1e-3
    n = 20000
    x, v = _gas(n, 1, L)
    prm = oracle.CouetteParams(L, dt, 500.0, RT, 0.0, 16)
    x1, vx, vy, vz, cell, nb, mg = oracle.move_couette(x, v[0], v[1], v[2], prm, 7, 3)
    free = x + v[0] * dt
    hits_closed = np.where(free < 0, np.floor(-free / L) + 1, np.floor(free / L)).astype(int)
    ok = hits_closed <= oracle.MAX_BOUNCES
    assert ok.mean() > 0.999 and hits_closed.max() >= 2
    y = np.mod(free, 2 * L)
    fold = np.where(y > L, 2 * L - y, y)
    assert np.allclose(x1[ok], fold[ok], rtol=0, atol=1e-12 * L)
    assert np.array_equal(nb[ok], hits_closed[ok])
    assert np.array_equal(vx[ok], np.where(hits_closed[ok] % 2 == 1, -v[0][ok], v[0][ok]))
    assert np.array_equal(vy, v[1]) and np.array_equal(vz, v[2])
    assert np.array_equal(cell[ok], np.minimum((fold[ok] * 16 / L).astype(int), 15))
    # particles that would need more hits than allowed are parked on a wall
    assert np.all((x1[~ok] == 0.0) | (x1[~ok] == L))


def test_no_wall_hit_is_plain_free_flight_and_margin_measures_the_decisions():
    L = 2.0
    x = np.array([0.5, 1.0, 1.9999, 0.25 + 1e-9])
    vx = np.array([100.0, -200.0, 0.0, 0.0])
    prm = oracle.CouetteParams(L, 1e-3, 500.0, RT, 1.0, 8)
    x1, vx1, vy1, vz1, cell, nb, mg = oracle.move_couette(x, vx, np.ones(4), np.ones(4), prm, 1, 0)
    assert np.allclose(x1, [0.6, 0.8, 1.9999, 0.25 + 1e-9], rtol=0, atol=1e-15)
    assert list(cell) == [2, 3, 7, 1] and list(nb) == [0, 0, 0, 0]
    assert np.allclose(mg, [0.05, 0.025, 0.0001 / 2.0, 1e-9 / 2.0], rtol=1e-6)
    assert np.array_equal(vx1, vx)


def test_diffuse_emission_has_the_flux_weighted_wall_maxwellian_moments():
    """Fully diffuse wall: normal speed Rayleigh-distributed (<vn> = sqrt(pi RT/2), <vn^2> = 2 RT), tangential
    components N(u_wall, RT) and N(0, RT) (Bird 1994, eq. 12.1-12.3 form); checked at 5 standard errors."""
    L, U, rt = 1.0, 500.0, 0.8 * RT
    n = 400000
    rng = np.random.default_rng(5)
    x = np.full(n, 1e-4)
    vx = -np.abs(rng.normal(0, math.sqrt(RT), n)) - 50.0  # all head for the lower wall
    prm = oracle.CouetteParams(L, 1e-5, U, rt, 1.0, 4)
    x1, vx1, vy1, vz1, cell, nb, mg = oracle.move_couette(x, vx, np.zeros(n), np.zeros(n), prm, 11, 2)
    hit = nb == 1
    assert hit.mean() > 0.99
    m = hit.sum()
    vn = vx1[hit]
    assert np.all(vn > 0)
    assert abs(vn.mean() - math.sqrt(math.pi * rt / 2)) < 5 * math.sqrt((2 - math.pi / 2) * rt / m)
    assert abs((vn**2).mean() - 2 * rt) < 5 * 2 * rt / math.sqrt(m)
    assert abs(vy1[hit].mean() + U) < 5 * math.sqrt(rt / m)  # lower wall moves with -U
    assert abs(vy1[hit].var() - rt) < 5 * rt * math.sqrt(2.0 / m)
    assert abs(vz1[hit].mean()) < 5 * math.sqrt(rt / m)
    assert abs(vz1[hit].var() - rt) < 5 * rt * math.sqrt(2.0 / m)
    assert abs(np.mean(vy1[hit] * vz1[hit])) < 5 * rt / math.sqrt(m)
    # the particle flies on with the new velocity for the rest of the step
    t_hit = (0.0 - x[hit]) / vx[hit]
    assert np.allclose(x1[hit], vn * (1e-5 - t_hit), rtol=1e-12, atol=0)
    # upper wall: mirrored normal, +U
    x = np.full(n, L - 1e-4)
    x1, vx1, vy1, vz1, cell, nb, mg = oracle.move_couette(x, -vx, np.zeros(n), np.zeros(n), prm, 11, 2)
    assert np.all(vx1[nb == 1] < 0) and abs(vy1[nb == 1].mean() - U) < 5 * math.sqrt(rt / m)


def test_partial_accommodation_fraction():
    n = 200000
    x = np.full(n, 1e-4)
    vx = np.full(n, -300.0)
    prm = oracle.CouetteParams(1.0, 1e-5, 500.0, RT, 0.3, 4)
    x1, vx1, vy1, vz1, cell, nb, mg = oracle.move_couette(x, vx, np.zeros(n), np.zeros(n), prm, 3, 0)
    spec = (vx1 == 300.0) & (vy1 == 0.0)
    assert abs((~spec).mean() - 0.3) < 5 * math.sqrt(0.3 * 0.7 / n)


def test_free_molecular_couette_shear_stress_and_temperature():
    """Collisionless gas between fully diffuse walls at +-U: each half-range population is the half Maxwellian of
    the wall it left, so <vx vy> = -U sqrt(2 RT / pi), <vy> = 0, <vy^2> = RT + U^2, <vx^2> = <vz^2> = RT, uniform
    density (free-molecular Couette flow, e.g. Bird 1994 section 7.4 / Kogan)."""
    L, U, dt = 1.0, 500.0, 1e-3
    n = 200000
    x, v = _gas(n, 9, L)
    prm = oracle.CouetteParams(L, dt, U, RT, 1.0, 10)
    vx, vy, vz = v
    touched = np.zeros(n, bool)
    for step in range(150):
        x, vx, vy, vz, cell, nb, mg = oracle.move_couette(x, vx, vy, vz, prm, 21, step)
        touched |= nb > 0
    assert touched.mean() > 0.97
    t = touched  # the few particles that never met a wall still carry the initial condition
    m = t.sum()
    sxy = math.sqrt(RT * (RT + U * U))
    assert abs(np.mean(vx[t] * vy[t]) + U * math.sqrt(2 * RT / math.pi)) < 5 * sxy / math.sqrt(m)
    assert abs(np.mean(vy[t] ** 2) - (RT + U * U)) < 0.02 * (RT + U * U)
    assert abs(np.mean(vz[t] ** 2) - RT) < 0.02 * RT
    assert abs(np.mean(vy[t])) < 5 * math.sqrt((RT + U * U) / m)
    assert np.all((x >= 0) & (x <= L))
    dens = np.bincount(cell, minlength=10) / n
    assert np.all(np.abs(dens - 0.1) < 5 * math.sqrt(0.1 * 0.9 / n))


def test_sample_cells_against_brute_force_and_accumulation():
    rng = np.random.default_rng(2)
    K, n = 7, 500
    cell = rng.integers(0, K, n)
    cell[cell == 3] = 4  # an empty cell
    rc, perm, cs = oracle.bin_particles(cell, K)
    v = rng.normal(0, 300.0, (3, n))[:, perm]
    acc = oracle.sample_cells(cs, v[0], v[1], v[2])
    cs_sorted = cell[perm]
    for k in range(K):
        sel = cs_sorted == k
        want = [sel.sum(), v[0][sel].sum(), v[1][sel].sum(), v[2][sel].sum(), (v[0][sel] ** 2).sum(),
                (v[1][sel] ** 2).sum(), (v[2][sel] ** 2).sum(), (v[0][sel] * v[1][sel]).sum()]
        assert np.allclose(acc[k], want, rtol=1e-12, atol=1e-9)
    acc2 = oracle.sample_cells(cs, v[0], v[1], v[2], acc.copy())
    assert np.allclose(acc2, 2 * acc, rtol=1e-14)

"""Pins for the CPU oracle (`oracle/`): closed forms, invariants, brute force, library special cases.

Pin numbers P1..P16 are those of SURVEY.md section 8(c) / DESIGN.md.  None of the expected
values here comes from the CUDA path, and none re-calls the oracle's own formula: brute force
is written out in numpy/pure Python in this file, library pins call scipy.ndimage.
"""
import itertools

import numpy as np
import pytest
from scipy import ndimage

import phantoms


def brute_moments(v, R):
    """Eq. (3) by explicit slicing: truncated cube, population variance."""
    nz, ny, nx = v.shape
    mean = np.zeros(v.shape)
    var = np.zeros(v.shape)
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        p = v[max(z - R, 0):z + R + 1, max(y - R, 0):y + R + 1, max(x - R, 0):x + R + 1].astype(np.float64)
        mean[z, y, x] = p.sum() / p.size
        var[z, y, x] = (p ** 2).sum() / p.size - (p.sum() / p.size) ** 2     # E(X^2) - E(X)^2, (A.4) PAPER.md:458
    return mean, var


# ---------------------------------------------------------------- moments
@pytest.mark.parametrize("shape", [(7, 6, 5), (4, 4, 4), (9, 1, 1), (1, 1, 9), (3, 8, 2)])
@pytest.mark.parametrize("R", [0, 1, 2, 3])
def test_P1_moments_brute_force(oracle_mod, shape, R):
    rng = np.random.default_rng(1)
    v = rng.uniform(-50, 50, size=shape).astype(np.float32)
    mean, var = oracle_mod.box_moments(v, R)
    bm, bv = brute_moments(v, R)
    np.testing.assert_allclose(mean, bm, rtol=0, atol=1e-10)
    np.testing.assert_allclose(var, bv, rtol=0, atol=1e-8)


def test_P1b_moments_hand_value(oracle_mod):
    # 3x3x3 cube holding 1..27: centre patch is the discrete uniform on 27 points:
    # mean 14, variance (27^2 - 1)/12.
    v = np.arange(1, 28, dtype=np.float32).reshape(3, 3, 3)
    mean, var = oracle_mod.box_moments(v, 1)
    assert mean[1, 1, 1] == 14.0
    assert abs(var[1, 1, 1] - (27 ** 2 - 1) / 12.0) < 1e-12
    # corner patch (0,0,0) holds the 8 values {1,2,4,5,10,11,13,14}
    corner = np.array([1, 2, 4, 5, 10, 11, 13, 14], dtype=np.float64)
    assert abs(mean[0, 0, 0] - corner.mean()) < 1e-12
    assert abs(var[0, 0, 0] - corner.var()) < 1e-12


def test_P2_moments_constant(oracle_mod):
    v = np.full((6, 7, 8), 1234.567, dtype=np.float32)
    mean, var = oracle_mod.box_moments(v, 3)
    assert np.all(mean == np.float64(np.float32(1234.567)))
    assert np.all(var == 0.0)


@pytest.mark.parametrize("R", [1, 3, 5])
def test_P3_moments_ramp_closed_form(oracle_mod, R):
    n = 2 * R + 5
    g = (1.5, -2.0, 0.25)
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    v = (g[0] * x + g[1] * y + g[2] * z).astype(np.float32)       # exactly representable
    mean, var = oracle_mod.box_moments(v, R)
    c = slice(R, n - R)
    np.testing.assert_allclose(mean[c, c, c], v[c, c, c], atol=1e-10)
    expect = (g[0] ** 2 + g[1] ** 2 + g[2] ** 2) * R * (R + 1) / 3.0   # variance of a discrete uniform on 2R+1 points, per axis
    np.testing.assert_allclose(var[c, c, c], expect, rtol=1e-12)


def test_golden_ramp_variance_and_paper_constants(oracle_mod):
    """tests/golden: the closed-form ramp variance table (Eq. 3) and the constants the paper prints."""
    import os
    gdir = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    rows = [ln.split() for ln in open(os.path.join(gdir, "ramp_variance.txt")) if ln.strip() and not ln.startswith("#")]
    g = (3.0, -2.0, 0.5)                                   # slopes along x, y, z
    n = 25
    z, y, x = np.meshgrid(np.arange(float(n)), np.arange(float(n)), np.arange(float(n)), indexing="ij")
    vol = (g[0] * x + g[1] * y + g[2] * z).astype(np.float32)
    c = n // 2
    for R_s, v_s in rows:
        R, per_unit = int(R_s), float(v_s)
        mean, var = oracle_mod.box_moments(vol, R)
        np.testing.assert_allclose(var[c, c, c], per_unit * sum(t * t for t in g), rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(mean[c, c, c], vol[c, c, c], rtol=1e-12)
    consts = {ln.split()[0]: ln.split()[1] for ln in open(os.path.join(gdir, "paper_constants.txt"))
              if ln.strip() and not ln.startswith("#")}
    assert float(consts["stop_eps"]) == 1.0e-4 and int(consts["stop_lag"]) == 10
    # the oracle's criterion uses exactly that lag: with eps = +inf it trips at k = 10, i.e. after 11 iterations
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(24, 20, 12))
    _, run, _ = oracle_mod.register_stop(ct, cbct, 1, 1.0, 1, 20, stop_eps=float("inf"))
    assert int(run[0]) == int(consts["stop_lag"]) + 1


def test_P4_moments_scipy_uniform_filter(oracle_mod):
    rng = np.random.default_rng(4)
    v = rng.normal(0, 100, size=(12, 11, 13)).astype(np.float32)
    R = 2
    mean, _ = oracle_mod.box_moments(v, R)
    box = ndimage.uniform_filter(v.astype(np.float64), 2 * R + 1, mode="constant")  # zero-padded mean over (2R+1)^3
    cnt = ndimage.uniform_filter(np.ones(v.shape), 2 * R + 1, mode="constant")       # in-volume fraction
    np.testing.assert_allclose(mean, box / cnt, atol=1e-9)


# ---------------------------------------------------------------- a, b and the correction
def test_P5_moment_matching_constraints(oracle_mod):
    """Eq. (4): with each voxel's own frozen (a, b), the transformed CBCT patch has the
    first two moments of the CT patch; and the oracle's s'(x) is a(x) I_s(x) + b(x)."""
    rng = np.random.default_rng(5)
    shape, R = (6, 7, 8), 2
    M = rng.normal(40, 30, size=shape).astype(np.float32)
    S = (0.7 * M + rng.normal(-100, 25, size=shape)).astype(np.float32)
    sp = oracle_mod.correct(S, M, R)
    for z, y, x in itertools.product(range(shape[0]), range(shape[1]), range(shape[2])):
        sl = (slice(max(z - R, 0), z + R + 1), slice(max(y - R, 0), y + R + 1), slice(max(x - R, 0), x + R + 1))
        pm, ps = M[sl].astype(np.float64), S[sl].astype(np.float64)
        a = pm.std() / ps.std()            # Eq. (5)
        b = pm.mean() - a * ps.mean()      # Eq. (6)
        t = a * ps + b
        assert abs(t.mean() - pm.mean()) < 1e-9                       # E(M) = E(S')
        assert abs((t ** 2).mean() - (pm ** 2).mean()) < 1e-6         # E(M^2) = E(S'^2)
        assert abs(sp[z, y, x] - (a * float(S[z, y, x]) + b)) < 2e-4   # fp32 output rounding only


def test_P6_identical_images_identity(oracle_mod):
    ct, _, _, _ = phantoms.make_pair(1, dims=(24, 20, 12))
    noisy = (ct + np.random.default_rng(6).normal(0, 5, ct.shape)).astype(np.float32)
    sp = oracle_mod.correct(noisy, noisy, 2)
    np.testing.assert_allclose(sp, noisy, atol=2e-4)
    # constant patches (sigma = 0): a = 0 and s' = mu_m = I_s
    flat = np.full((5, 5, 5), -1000.0, dtype=np.float32)
    assert np.array_equal(oracle_mod.correct(flat, flat, 1), flat)


def test_P7_affine_cbct_is_corrected_exactly(oracle_mod):
    rng = np.random.default_rng(7)
    ct = rng.normal(0, 200, size=(8, 9, 10)).astype(np.float32)
    cbct = (0.9 * ct.astype(np.float64) - 150.0).astype(np.float32)
    sp = oracle_mod.correct(cbct, ct, 2)
    np.testing.assert_allclose(sp, ct, atol=2e-3)       # cbct itself is rounded to fp32
    # negative gain is NOT undone: a >= 0 by construction
    neg = (-0.9 * ct.astype(np.float64)).astype(np.float32)
    assert np.abs(oracle_mod.correct(neg, ct, 2) - ct).max() > 50.0


def test_P8_static_affine_invariance(oracle_mod):
    """correct(alpha*cbct + beta, m) = correct(cbct, m): the global Delta-HU shift is a no-op here."""
    rng = np.random.default_rng(8)
    m = rng.normal(0, 100, size=(7, 8, 9)).astype(np.float32)
    s = rng.normal(50, 80, size=(7, 8, 9)).astype(np.float32)
    s2 = (2.0 * s + 128.0).astype(np.float32)            # exact in fp32 for these magnitudes? power-of-two gain: yes up to rounding of +128
    a = oracle_mod.correct(s, m, 2)
    b = oracle_mod.correct(s2, m, 2)
    np.testing.assert_allclose(a, b, atol=2e-3)


def test_var_s_zero_gives_mu_m(oracle_mod):
    m = np.random.default_rng(9).normal(0, 10, size=(5, 5, 5)).astype(np.float32)
    s = np.full((5, 5, 5), 77.0, dtype=np.float32)
    mean, _ = oracle_mod.box_moments(m, 1)
    np.testing.assert_allclose(oracle_mod.correct(s, m, 1), mean, atol=1e-5)
    # R = 0: var = 0 everywhere -> s' = m
    assert np.array_equal(oracle_mod.correct(s, m, 0), m)


# ---------------------------------------------------------------- warp
def test_P9_warp(oracle_mod):
    rng = np.random.default_rng(10)
    I = rng.normal(0, 300, size=(9, 10, 11)).astype(np.float32)
    zero = np.zeros((3,) + I.shape, dtype=np.float32)
    assert np.array_equal(oracle_mod.warp(I, zero), I)                     # identity, bit exact
    sh = zero.copy(); sh[0] = 2; sh[1] = -1; sh[2] = 1                      # integer shift (x+2, y-1, z+1)
    w = oracle_mod.warp(I, sh)
    assert np.array_equal(w[0:8, 1:10, 0:9], I[1:9, 0:9, 2:11])
    # trilinear reproduces affine functions: out(x) = g.(x + r(x)) for in-range samples
    z, y, x = np.meshgrid(np.arange(9.), np.arange(10.), np.arange(11.), indexing="ij")
    ramp = (3 * x - 2 * y + 0.5 * z).astype(np.float32)
    r = rng.uniform(-1.5, 1.5, size=(3,) + I.shape).astype(np.float32)
    px, py, pz = x + r[0], y + r[1], z + r[2]
    inside = (px >= 0) & (px <= 10) & (py >= 0) & (py <= 9) & (pz >= 0) & (pz <= 8)
    w = oracle_mod.warp(ramp, r)
    np.testing.assert_allclose(w[inside], (3 * px - 2 * py + 0.5 * pz)[inside], atol=1e-4)
    # library special case: map_coordinates(order=1) at the clamped coordinates
    coords = np.stack([np.clip(pz, 0, 8), np.clip(py, 0, 9), np.clip(px, 0, 10)])
    ref = ndimage.map_coordinates(I.astype(np.float64), coords, order=1, mode="nearest")
    np.testing.assert_allclose(oracle_mod.warp(I, r), ref, atol=1e-3)
    # axis of length 1: weight 0 along it
    thin = rng.normal(size=(1, 4, 5)).astype(np.float32)
    rz = np.zeros((3, 1, 4, 5), dtype=np.float32); rz[2] = 0.7
    assert np.array_equal(oracle_mod.warp(thin, rz), thin)


# ---------------------------------------------------------------- force
def test_P10_force(oracle_mod):
    rng = np.random.default_rng(11)
    shape = (6, 7, 8)
    s = rng.normal(0, 100, size=shape).astype(np.float32)
    r0 = rng.normal(0, 1, size=(3,) + shape).astype(np.float32)
    assert np.array_equal(oracle_mod.force_update(s, s, r0), r0)                       # m = s' -> dr = 0
    flat = np.full(shape, 5.0, dtype=np.float32)
    assert np.array_equal(oracle_mod.force_update(s, flat, r0), r0)                    # grad s' = 0 -> dr = 0
    m = rng.normal(0, 100, size=shape).astype(np.float32)
    dr = oracle_mod.force_update(m, s, np.zeros_like(r0))
    assert np.sqrt((dr.astype(np.float64) ** 2).sum(0)).max() <= 0.5 + 1e-6            # |dr| <= 1/2 (AM-GM)
    # ramp: s' = g x, m = s' - g*delta  ->  true shift +delta along x, |dr| = delta/(1+delta^2), slope independent
    z, y, x = np.meshgrid(np.arange(6.), np.arange(7.), np.arange(8.), indexing="ij")
    for g, delta in ((10.0, 0.5), (200.0, 2.0), (-30.0, 0.25)):
        sp = (g * x).astype(np.float32)
        mm = (g * x - g * delta).astype(np.float32)
        d = oracle_mod.force_update(mm, sp, np.zeros_like(r0), eps_den=0.0)
        inner = d[:, :, :, 1:-1]
        np.testing.assert_allclose(inner[0], delta / (1 + delta ** 2), rtol=1e-6)     # sign: + (descends for pull-back warp)
        assert np.all(inner[1] == 0) and np.all(inner[2] == 0)
    # central difference with clamped indices: border gets half the one-sided difference
    sp = (10.0 * x).astype(np.float32)
    d = oracle_mod.force_update(sp - 5.0, sp, np.zeros_like(r0), eps_den=0.0)
    gb, dd = 5.0, 5.0
    np.testing.assert_allclose(d[0, :, :, 0], dd * gb / (gb * gb + dd * dd), rtol=1e-6)


def test_double_force_pins(oracle_mod):
    """NEXT-2, both terms of Eq. (1): closed forms and symmetries, none re-typing the formula."""
    rng = np.random.default_rng(12)
    shape = (6, 7, 8)
    s = rng.normal(0, 100, size=shape).astype(np.float32)
    m = rng.normal(0, 100, size=shape).astype(np.float32)
    r0 = rng.normal(0, 1, size=(3,) + shape).astype(np.float32)
    zero = np.zeros_like(r0)
    f2 = lambda mm, ss, r, **kw: oracle_mod.force_update(mm, ss, r, double_force=True, **kw)
    assert np.array_equal(f2(s, s, r0), r0)                                            # m = s' -> dr = 0
    # a flat moving image has no active force: the double force reduces to the Thirion force ...
    flat = np.full(shape, 5.0, dtype=np.float32)
    assert np.array_equal(f2(flat, s, zero), oracle_mod.force_update(flat, s, zero))
    # ... and a flat static image leaves ONLY the active term = the Thirion force with the roles swapped, negated
    np.testing.assert_allclose(f2(m, flat, zero), -oracle_mod.force_update(flat, m, zero), rtol=1e-6, atol=1e-7)
    # exchanging the two images negates the double force exactly (each term maps onto the other)
    assert np.array_equal(f2(m, s, zero), -f2(s, m, zero))
    # each term is bounded by 1/2 (AM-GM) -> |dr| <= 1
    d = f2(m, s, zero)
    assert np.sqrt((d.astype(np.float64) ** 2).sum(0)).max() <= 1.0 + 1e-6
    # ramp: s' = g x, m = s' - g delta: both gradients equal g -> twice the single force, 2 delta / (1 + delta^2)
    z, y, x = np.meshgrid(np.arange(6.), np.arange(7.), np.arange(8.), indexing="ij")
    for g, delta in ((10.0, 0.5), (200.0, 2.0), (-30.0, 0.25)):
        sp = (g * x).astype(np.float32)
        mm = (g * x - g * delta).astype(np.float32)
        d = f2(mm, sp, zero, eps_den=0.0)[:, :, :, 1:-1]
        np.testing.assert_allclose(d[0], 2 * delta / (1 + delta ** 2), rtol=1e-6)
        assert np.all(d[1] == 0) and np.all(d[2] == 0)
    # different slopes: s' = g x, m = h x - c  ->  d g/(g^2+d^2) + d h/(h^2+d^2) with d = s' - m evaluated per voxel
    g, h, c = 12.0, 7.0, 3.0
    sp, mm = (g * x).astype(np.float32), (h * x - c).astype(np.float32)
    dd = (g - h) * x[:, :, 1:-1] + c
    want = dd * g / (g * g + dd * dd) + dd * h / (h * h + dd * dd)
    np.testing.assert_allclose(f2(mm, sp, zero, eps_den=0.0)[0, :, :, 1:-1], want, rtol=1e-6)


def test_double_force_recovers_a_translation(oracle_mod):
    """whole loop with the double force: same sign convention as P11, converges at least as far as the single force"""
    ct, _, _, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    u = np.zeros((3,) + ct.shape, dtype=np.float32); u[0], u[1], u[2] = 2.0, -1.0, 1.0
    target = phantoms.pullback(ct, u)
    rng = np.random.default_rng(5)
    cbct = (0.9 * target + rng.normal(0, 20, ct.shape)).astype(np.float32)
    rmse = lambda r: float(np.sqrt(np.mean((oracle_mod.warp(ct, r) - target) ** 2)))
    r1, _ = oracle_mod.register(ct, cbct, 3, 1.5, 1, 40, want_corr=False)
    r2, _ = oracle_mod.register(ct, cbct, 3, 1.5, 1, 40, want_corr=False, double_force=True)
    e0, e1, e2 = rmse(np.zeros_like(u)), rmse(r1), rmse(r2)
    assert e2 < e0 / 2.5 and e2 < 1.1 * e1, (e0, e1, e2)


def test_convergence_measure_pins(oracle_mod):
    """NEXT-3: l = sum|dr| / sum|r|.  Closed form on a ramp, Euclidean norm per voxel (reading A16)."""
    nz, ny, nx = 4, 5, 9
    z, y, x = np.meshgrid(np.arange(float(nz)), np.arange(float(ny)), np.arange(float(nx)), indexing="ij")
    g, delta = 20.0, 0.75
    sp, mm = (g * x).astype(np.float32), (g * x - g * delta).astype(np.float32)
    r = np.empty((3, nz, ny, nx), dtype=np.float32); r[0], r[1], r[2] = 3.0, -4.0, 12.0      # |r| = 13 at every voxel
    sdr, sr = oracle_mod.force_norms(mm, sp, r, eps_den=0.0)
    d = g * delta
    inner, border = d * g / (g * g + d * d), d * (g / 2) / ((g / 2) ** 2 + d * d)             # clamped central difference
    np.testing.assert_allclose(sdr, nz * ny * ((nx - 2) * inner + 2 * border), rtol=1e-6)
    np.testing.assert_allclose(sr, 13.0 * nz * ny * nx, rtol=1e-12)
    # a diagonal ramp: |dr| is the Euclidean norm, not the sum of |components|
    sp2 = (g * (x + y)).astype(np.float32)
    sdr2, _ = oracle_mod.force_norms(sp2 - np.float32(d), sp2, r, eps_den=0.0)
    core = (slice(1, -1),) * 3
    per_voxel = np.sqrt(2.0) * d * g / (2 * g * g + d * d)
    one, _ = oracle_mod.force_norms((sp2 - np.float32(d))[core], sp2[core], r[(slice(None),) + core], eps_den=0.0)
    assert sdr2 > 0 and one > 0
    dr = oracle_mod.force_update(sp2 - np.float32(d), sp2, np.zeros_like(r), eps_den=0.0)
    np.testing.assert_allclose(np.sqrt((dr.astype(np.float64) ** 2).sum(0))[core], per_voxel, rtol=1e-5)
    np.testing.assert_allclose(sdr2, np.sqrt((dr.astype(np.float64) ** 2).sum(0)).sum(), rtol=1e-6)
    # double force: both terms equal on equal slopes -> twice the sum
    sdr_d, _ = oracle_mod.force_norms(mm, sp, r, eps_den=0.0, double_force=True)
    np.testing.assert_allclose(sdr_d, 2 * sdr, rtol=1e-6)


def test_stopping_criterion_pins(oracle_mod):
    """NEXT-3: stop at the first k >= 10 with l(k-10) - l(k) <= eps, inside each level; the iteration that trips it is
    completed; an early-stopped run IS the fixed-count run with those counts."""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    R, sigma, levels, iters, eps = 3, 1.5, 2, 40, 2e-3
    r, run, lt = oracle_mod.register_stop(ct, cbct, R, sigma, levels, iters, stop_eps=eps)
    assert run.min() >= 11 and run.min() < iters                      # never before 11 iterations; something stopped early
    for lev in range(levels):
        row, n = lt[levels - 1 - lev], int(run[lev])
        assert np.all(np.isfinite(row[1:n])) and np.all(np.isnan(row[n:]))
        diffs = row[:n - 10] - row[10:n]                              # criterion values for k = 10 .. n-1
        if n < iters:
            assert diffs[-1] <= eps and np.all(diffs[:-1] > eps)      # tripped at k = n-1 and not before
        else:
            assert np.all(diffs[:-1] > eps)
    assert np.isinf(lt[0, 0])                                         # r = 0 at the coarsest level's first iteration
    # l itself, recomputed from the stepwise functions for the first two iterations of the coarsest level
    c, b = oracle_mod.downsample(ct), oracle_mod.downsample(cbct)
    rr = np.zeros((3,) + c.shape, dtype=np.float32)
    for k in range(2):
        m = oracle_mod.warp(c, rr)
        sp = oracle_mod.correct(b, m, R)
        dr = oracle_mod.force_update(m, sp, np.zeros_like(rr))
        num = np.sqrt((dr.astype(np.float64) ** 2).sum(0)).sum()
        den = np.sqrt((rr.astype(np.float64) ** 2).sum(0)).sum()
        if den > 0:
            np.testing.assert_allclose(lt[0, k], num / den, rtol=1e-5)
        rr = oracle_mod.demons_step(m, sp, rr, sigma)
    # composition: the same counts as a fixed schedule give the same field, bit for bit; and stop_eps = None runs them all
    r_fixed, run_fixed, _ = oracle_mod.register_stop(ct, cbct, R, sigma, levels, iters, iters_per_level=run)
    assert np.array_equal(r, r_fixed) and np.array_equal(run, run_fixed)
    r_all, run_all, _ = oracle_mod.register_stop(ct, cbct, R, sigma, levels, 12)
    r_ref, _ = oracle_mod.register(ct, cbct, R, sigma, levels, 12, want_corr=False)
    assert np.array_equal(r_all, r_ref) and np.all(run_all == 12)


def test_force_components_and_axes(oracle_mod):
    """each component uses its own axis' gradient (catches transposed strides)."""
    z, y, x = np.meshgrid(np.arange(5.), np.arange(6.), np.arange(7.), indexing="ij")
    zero = np.zeros((3, 5, 6, 7), dtype=np.float32)
    for c, coord in enumerate((x, y, z)):
        sp = (8.0 * coord).astype(np.float32)
        d = oracle_mod.force_update(sp - 8.0, sp, zero, eps_den=0.0)
        core = d[:, 1:-1, 1:-1, 1:-1]
        np.testing.assert_allclose(core[c], 0.5, rtol=1e-6)
        for o in range(3):
            if o != c:
                assert np.all(core[o] == 0)


# ---------------------------------------------------------------- Gaussian
@pytest.mark.parametrize("sigma", [1.0, 1.5, 2.0, 3.0])
def test_P14_gaussian(oracle_mod, sigma):
    w = oracle_mod.gauss_weights(sigma).astype(np.float64)
    K = int(np.ceil(3 * sigma))
    assert w.size == 2 * K + 1
    assert abs(w.sum() - 1.0) < 1e-6 and np.allclose(w, w[::-1])
    # library: scipy's own truncated, normalised Gaussian kernel via an impulse
    imp = np.zeros(4 * K + 1); imp[2 * K] = 1.0
    ref = ndimage.gaussian_filter1d(imp, sigma, truncate=K / sigma + 1e-9, mode="nearest")[K:3 * K + 1]
    np.testing.assert_allclose(w, ref, atol=1e-7)
    n = 2 * K + 6
    const = np.full((3, n, n + 1, n + 2), 0.0, dtype=np.float32); const[0] = 1.25; const[1] = -3.5; const[2] = 7.0
    out = oracle_mod.smooth_field(const, sigma)
    np.testing.assert_allclose(out, const, atol=1e-6)                                  # constant preserved
    # impulse response = outer product of the 1-D kernel
    f = np.zeros((3, 2 * K + 1, 2 * K + 1, 2 * K + 1), dtype=np.float32); f[1, K, K, K] = 1.0
    out = oracle_mod.smooth_field(f, sigma)
    np.testing.assert_allclose(out[1], np.einsum("i,j,k->ijk", w, w, w), atol=1e-7)
    assert np.all(out[0] == 0) and np.all(out[2] == 0)
    # linear ramp unchanged >= K from the border
    z, y, x = np.meshgrid(np.arange(n), np.arange(n + 1), np.arange(n + 2), indexing="ij")
    ramp = np.stack([0.1 * x - 0.2 * y + 0.05 * z] * 3).astype(np.float32)
    out = oracle_mod.smooth_field(ramp, sigma)
    c = (slice(None), slice(K, n - K), slice(K, n + 1 - K), slice(K, n + 2 - K))
    np.testing.assert_allclose(out[c], ramp[c], atol=2e-6)
    # library: three convolve1d passes with replicate border
    rng = np.random.default_rng(14)
    fld = rng.normal(0, 2, size=(3, 9, 10, 11)).astype(np.float32)
    ref = fld.astype(np.float64)
    for ax in (3, 2, 1):
        ref = ndimage.convolve1d(ref, w, axis=ax, mode="nearest")
    np.testing.assert_allclose(oracle_mod.smooth_field(fld, sigma), ref, atol=1e-5)


# ---------------------------------------------------------------- pyramid
def test_P15_pyramid(oracle_mod):
    const = np.full((4, 6, 8), 3.25, dtype=np.float32)
    assert np.all(oracle_mod.downsample(const) == 3.25)
    z, y, x = np.meshgrid(np.arange(4.), np.arange(6.), np.arange(8.), indexing="ij")
    ramp = (2 * x - 3 * y + 5 * z).astype(np.float32)
    d = oracle_mod.downsample(ramp)
    zc, yc, xc = np.meshgrid(np.arange(2.), np.arange(3.), np.arange(4.), indexing="ij")
    np.testing.assert_allclose(d, 2 * (2 * xc + 0.5) - 3 * (2 * yc + 0.5) + 5 * (2 * zc + 0.5), atol=1e-5)
    rng = np.random.default_rng(15)
    v = rng.normal(size=(4, 6, 8)).astype(np.float32)
    np.testing.assert_allclose(oracle_mod.downsample(v), v.reshape(2, 2, 3, 2, 4, 2).mean(axis=(1, 3, 5)), atol=1e-6)
    c = np.zeros((3, 3, 4, 5), dtype=np.float32); c[0] = 1.0; c[1] = -2.0; c[2] = 0.5
    up = oracle_mod.upsample_field(c)
    assert up.shape == (3, 6, 8, 10)
    assert np.all(up[0] == 2.0) and np.all(up[1] == -4.0) and np.all(up[2] == 1.0)       # constant c -> 2c
    # r = g * i_coarse  ->  g * i_fine - g/2 in the interior (coarse cell centre i sits at fine 2i + 1/2)
    zc, yc, xc = np.meshgrid(np.arange(3.), np.arange(4.), np.arange(5.), indexing="ij")
    g = 0.75
    rc = np.stack([g * xc, g * yc, g * zc]).astype(np.float32)
    up = oracle_mod.upsample_field(rc)
    zf, yf, xf = np.meshgrid(np.arange(6.), np.arange(8.), np.arange(10.), indexing="ij")
    inner = (slice(1, -1), slice(1, -1), slice(1, -1))
    np.testing.assert_allclose(up[0][inner], (g * xf - g / 2)[inner], atol=1e-6)
    np.testing.assert_allclose(up[1][inner], (g * yf - g / 2)[inner], atol=1e-6)
    np.testing.assert_allclose(up[2][inner], (g * zf - g / 2)[inner], atol=1e-6)


# ---------------------------------------------------------------- symmetry (indexing)
def _one_iteration(o, ct, cbct, r, R, sigma):
    m = o.warp(ct, r)
    sp = o.correct(cbct, m, R)
    return o.demons_step(m, sp, r, sigma), sp


def test_P16_flip_and_permute_equivariance(oracle_mod):
    rng = np.random.default_rng(16)
    shape = (6, 8, 10)
    ct = ndimage.gaussian_filter(rng.normal(0, 300, size=shape), 1.0).astype(np.float32)
    cbct = (0.9 * ndimage.shift(ct, (0.4, -0.6, 0.8), order=1, mode="nearest") + rng.normal(0, 5, shape)).astype(np.float32)
    r0 = rng.normal(0, 0.3, size=(3,) + shape).astype(np.float32)
    r1, sp1 = _one_iteration(oracle_mod, ct, cbct, r0, 1, 1.0)
    for axis_np, comp in ((2, 0), (1, 1), (0, 2)):             # numpy axis 2 = x = component 0
        rf = np.flip(r0, axis=axis_np + 1).copy(); rf[comp] = -rf[comp]
        r2, sp2 = _one_iteration(oracle_mod, np.flip(ct, axis_np).copy(), np.flip(cbct, axis_np).copy(), rf, 1, 1.0)
        back = np.flip(r2, axis=axis_np + 1).copy(); back[comp] = -back[comp]
        np.testing.assert_allclose(back, r1, atol=2e-6)
        np.testing.assert_allclose(np.flip(sp2, axis_np), sp1, atol=2e-3)
    # swap x and z (numpy axes 2 and 0): components 0 and 2 swap
    rt = np.ascontiguousarray(r0.transpose(0, 3, 2, 1))[[2, 1, 0]]
    r2, sp2 = _one_iteration(oracle_mod, np.ascontiguousarray(ct.transpose(2, 1, 0)),
                             np.ascontiguousarray(cbct.transpose(2, 1, 0)), np.ascontiguousarray(rt), 1, 1.0)
    np.testing.assert_allclose(r2[[2, 1, 0]].transpose(0, 3, 2, 1), r1, atol=2e-6)
    np.testing.assert_allclose(sp2.transpose(2, 1, 0), sp1, atol=2e-3)


# ---------------------------------------------------------------- whole loop
def _edge_normal_error(ct, r, u):
    """mean |(r - u).n| where n = grad(ct)/|grad(ct)| at strong edges (the recoverable component)."""
    gz, gy, gx = np.gradient(ct.astype(np.float64))
    mag = np.sqrt(gx ** 2 + gy ** 2 + gz ** 2)
    sel = mag > np.percentile(mag, 95)
    n = np.stack([gx, gy, gz]) / np.maximum(mag, 1e-9)
    err = np.abs(((r - u) * n).sum(0))[sel].mean()
    ref = np.abs((u * n).sum(0))[sel].mean()
    return err, ref


def test_P11_translation_is_recovered_with_the_documented_sign(oracle_mod):
    ct, _, _, p = phantoms.make_pair(1)
    rng = np.random.default_rng(111)
    u = np.zeros((3,) + ct.shape, dtype=np.float32); u[0] = 2.0; u[1] = -1.0; u[2] = 1.0
    cbct = phantoms.make_cbct(ct, u, rng, gain=0.9, cupping=150.0, noise=20.0)
    target = phantoms.pullback(ct, u)
    r, corr = oracle_mod.register(ct, cbct, R=3, sigma=1.5, levels=1, iters=50)
    rmse0 = np.sqrt(np.mean((ct - target) ** 2))
    rmse1 = np.sqrt(np.mean((oracle_mod.warp(ct, r) - target) ** 2))
    assert rmse1 < rmse0 / 3.0, (rmse0, rmse1)
    err, ref = _edge_normal_error(ct, r, u)
    assert err < 0.4 and err < 0.5 * ref, (err, ref)
    # and the opposite convention would have diverged: the recovered field points along +u at edges
    gz, gy, gx = np.gradient(ct.astype(np.float64))
    mag = np.sqrt(gx ** 2 + gy ** 2 + gz ** 2)
    sel = mag > np.percentile(mag, 95)
    n = np.stack([gx, gy, gz]) / np.maximum(mag, 1e-9)
    assert np.mean(((r * n).sum(0) * (u * n).sum(0))[sel]) > 0


def test_P12_sinusoid_config1(oracle_mod):
    ct, cbct, u, p = phantoms.make_pair(1)
    target = phantoms.pullback(ct, u)
    r, corr, trace = oracle_mod.register(ct, cbct, p["patch_radius"], p["sigma"], p["levels"], p["iters"], want_trace=True)
    rmse0 = np.sqrt(np.mean((ct - target) ** 2))
    rmse1 = np.sqrt(np.mean((oracle_mod.warp(ct, r) - target) ** 2))
    assert rmse1 < rmse0 / 2.5, (rmse0, rmse1)
    # the corrected CBCT takes the deformed CT's intensity distribution
    warped = oracle_mod.warp(ct, r)
    assert np.sqrt(np.mean((corr - warped) ** 2)) < 0.5 * np.sqrt(np.mean((cbct - warped) ** 2))
    assert np.all(np.isfinite(trace)) and trace[-1] > 0
    # out_corr = correct(cbct, warp(ct, out_disp)) (reading A12)
    np.testing.assert_array_equal(corr, oracle_mod.correct(cbct, warped, p["patch_radius"]))


def test_P13_fixed_point(oracle_mod):
    """cbct = alpha*ct + beta, r0 = 0 is a fixed point ("identical images give zero force").

    With inputs for which the affine map is exact in fp32 (integer HU, alpha = 1/2) the correction returns
    ct to fp64 rounding (bit-exactly unless ct = 0), so |r| stays < 1e-12 for every iteration and level.  With alpha = 0.9 the
    fp32 rounding of cbct leaves |d| ~ 1e-4 HU and the first iteration moves r by < 1e-4 voxel; on a
    noise-free pair that residue is then amplified in flat regions (the demons force is invariant to the
    intensity scale) -- DESIGN.md "Findings", the reason the paper masks a."""
    ct, _, _, _ = phantoms.make_pair(1, dims=(32, 32, 16))
    cti = np.round(ct).astype(np.float32)
    cbct = (0.5 * cti - 120.0).astype(np.float32)
    assert np.array_equal(cbct.astype(np.float64), 0.5 * cti.astype(np.float64) - 120.0)
    r, corr = oracle_mod.register(cti, cbct, R=2, sigma=1.5, levels=2, iters=10)
    assert np.abs(r).max() < 1e-12        # not exactly 0 only where ct == 0 (s' = 1e-14 instead of 0)
    np.testing.assert_allclose(corr, cti, rtol=0, atol=1e-10)
    cbct9 = (0.9 * ct.astype(np.float64) - 120.0).astype(np.float32)
    r, _ = oracle_mod.register(ct, cbct9, R=2, sigma=1.5, levels=1, iters=1)
    assert np.abs(r).max() < 2e-4


def test_multilevel_register_matches_stepwise_composition(oracle_mod):
    """oracle_register is exactly the documented composition of the step functions (levels, order, up-sampling)."""
    ct, cbct, u, _ = phantoms.make_pair(1, dims=(32, 24, 16))
    R, sigma, iters = 2, 1.5, 3
    r, corr = oracle_mod.register(ct, cbct, R, sigma, levels=2, iters=iters)
    ct1, cb1 = oracle_mod.downsample(ct), oracle_mod.downsample(cbct)
    rr = np.zeros((3,) + ct1.shape, dtype=np.float32)
    for _ in range(iters):
        m = oracle_mod.warp(ct1, rr); rr = oracle_mod.demons_step(m, oracle_mod.correct(cb1, m, R), rr, sigma)
    rr = oracle_mod.upsample_field(rr)
    for _ in range(iters):
        m = oracle_mod.warp(ct, rr); rr = oracle_mod.demons_step(m, oracle_mod.correct(cbct, m, R), rr, sigma)
    np.testing.assert_array_equal(r, rr)
    np.testing.assert_array_equal(corr, oracle_mod.correct(cbct, oracle_mod.warp(ct, rr), R))

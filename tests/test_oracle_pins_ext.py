"""Pins for the oracle functions added for SURVEY.md section 8(f) and for the full-size checks:
the `_at` samplers, per-axis patch radii and pyramid factors (NEXT-4), the summed-area moments, the mask and the
interpolation of a, b (NEXT-1), the Fig.-9 diagnostics and the general driver `register_ex`.

As in test_oracle_pins.py: no expected value comes from the CUDA path and none re-calls the oracle's own
formula -- brute force is written out here in numpy / pure Python, closed forms are derived in the comments.
"""
import itertools
import math

import numpy as np
import pytest

import phantoms


def brute_moments3(v, R):
    """Eq. (3) by explicit slicing: truncated box of per-axis radius R = (Rx, Ry, Rz)."""
    nz, ny, nx = v.shape
    mean = np.zeros(v.shape)
    var = np.zeros(v.shape)
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        p = v[max(z - R[2], 0):z + R[2] + 1, max(y - R[1], 0):y + R[1] + 1, max(x - R[0], 0):x + R[0] + 1].astype(np.float64)
        mean[z, y, x] = p.sum() / p.size
        var[z, y, x] = (p ** 2).sum() / p.size - (p.sum() / p.size) ** 2
    return mean, var


# ---------------------------------------------------------------- the samplers used by the full-size checks
@pytest.mark.parametrize("R", [0, 1, 3])
def test_at_samplers_decode_indices_like_the_full_loops(oracle_mod, R):
    """box_moments_at / correct_at on EVERY index of a non-square volume (nx != ny != nz, so an x/y/z mix-up in the
    index decode cannot cancel) equal the whole-volume functions bit for bit; and the whole-volume function is
    itself pinned by brute force (P1), so is the decode."""
    rng = np.random.default_rng(5)
    shape = (5, 7, 9)                                         # nz, ny, nx
    v = rng.uniform(-300, 900, size=shape).astype(np.float32)
    m = rng.uniform(-300, 900, size=shape).astype(np.float32)
    idx = np.arange(v.size, dtype=np.int64)
    mean, var = oracle_mod.box_moments(v, R)
    mean_at, var_at = oracle_mod.box_moments_at(v, R, idx)
    assert np.array_equal(mean_at, mean.ravel()) and np.array_equal(var_at, var.ravel())
    corr = oracle_mod.correct(v, m, R)
    corr_at = oracle_mod.correct_at(v, m, R, idx)
    assert np.array_equal(corr_at.astype(np.float32), corr.ravel())
    # a permuted, repeated subset keeps the order of the request
    sub = rng.integers(0, v.size, 40)
    assert np.array_equal(oracle_mod.box_moments_at(v, R, sub)[0], mean.ravel()[sub])
    # brute force at three hand-decoded voxels: idx = (z*ny + y)*nx + x
    bm, bv = brute_moments3(v, (R, R, R))
    for z, y, x in [(0, 0, 8), (4, 6, 0), (2, 3, 5)]:
        i = np.array([(z * 7 + y) * 9 + x])
        mu_i, var_i = oracle_mod.box_moments_at(v, R, i)
        assert abs(mu_i[0] - bm[z, y, x]) < 1e-10 and abs(var_i[0] - bv[z, y, x]) < 1e-7


# ---------------------------------------------------------------- NEXT-4: per-axis radius
@pytest.mark.parametrize("R", [(1, 1, 1), (2, 1, 0), (0, 3, 1), (3, 3, 1), (1, 2, 3)])
def test_moments3_brute_force(oracle_mod, R):
    rng = np.random.default_rng(2)
    v = rng.uniform(-50, 50, size=(5, 6, 8)).astype(np.float32)
    mean, var = oracle_mod.box_moments3(v, R)
    bm, bv = brute_moments3(v, R)
    np.testing.assert_allclose(mean, bm, rtol=0, atol=1e-10)
    np.testing.assert_allclose(var, bv, rtol=0, atol=1e-8)
    if R[0] == R[1] == R[2]:
        m0, v0 = oracle_mod.box_moments(v, R[0])
        assert np.array_equal(m0, mean) and np.array_equal(v0, var)


def test_moments3_anisotropic_ramp_closed_form(oracle_mod):
    """linear ramp: interior variance = sum_c g_c^2 R_c (R_c + 1) / 3 (a discrete uniform on 2 R_c + 1 points per axis)."""
    g = (1.5, -2.0, 0.25)
    for R in [(12, 12, 3), (1, 1, 1), (5, 5, 1), (2, 4, 0)]:     # 25x25x7 is the paper's largest patch
        n = [2 * r + 3 for r in R]
        z, y, x = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
        v = (g[0] * x + g[1] * y + g[2] * z).astype(np.float32)
        mean, var = oracle_mod.box_moments3(v, R)
        c = (slice(R[2], n[2] - R[2]), slice(R[1], n[1] - R[1]), slice(R[0], n[0] - R[0]))
        expect = sum(g[i] ** 2 * R[i] * (R[i] + 1) / 3.0 for i in range(3))
        np.testing.assert_allclose(var[c], expect, rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(mean[c], v[c], atol=1e-10)


# ---------------------------------------------------------------- exact (128-bit integer) summed-area moments vs the naive loops
@pytest.mark.parametrize("shape", [(7, 6, 5), (4, 4, 4), (9, 1, 1), (1, 1, 9), (3, 8, 2)])
@pytest.mark.parametrize("R", [0, 1, 2, 3, (3, 1, 2)])
def test_sat_moments_match_naive(oracle_mod, shape, R):
    rng = np.random.default_rng(3)
    v = rng.uniform(-50, 50, size=shape).astype(np.float32)
    mean, var = oracle_mod.box_moments3(v, R)
    ms, vs = oracle_mod.box_moments3(v, R, sat=True)
    np.testing.assert_allclose(ms, mean, rtol=0, atol=1e-9)
    np.testing.assert_allclose(vs, var, rtol=0, atol=1e-9)
    bm, bv = brute_moments3(v, (R, R, R) if np.isscalar(R) else R)
    np.testing.assert_allclose(ms, bm, rtol=0, atol=1e-9)
    np.testing.assert_allclose(vs, bv, rtol=0, atol=1e-8)


def test_sat_moments_refuse_values_outside_their_range(oracle_mod):
    """the fixed-point tables hold |v| < 2^14 HU: anything else is an error, not silently unwritten outputs; the driver
    falls back to the naive loops (same result as without the policy)"""
    v = np.zeros((4, 5, 6), dtype=np.float32)
    for bad in (16384.0, -3e4, np.inf, np.nan):
        v[1, 2, 3] = bad
        with pytest.raises(ValueError):
            oracle_mod.box_moments3(v, 1, sat=True)
    rng = np.random.default_rng(5)
    ct = rng.normal(0, 100, size=(8, 8, 8)).astype(np.float32)
    cbct = ct + rng.normal(0, 20, size=ct.shape).astype(np.float32)
    ct[0, 0, 0] = 20000.0
    a = oracle_mod.register_ex(ct, cbct, 1, 1.0, 1, 4, sat_between=True)
    b = oracle_mod.register_ex(ct, cbct, 1, 1.0, 1, 4)
    assert np.array_equal(a["disp"], b["disp"])


def test_sat_moments_on_a_phantom(oracle_mod):
    """HU-scale data with large flat regions: the summed-area route is exact integer arithmetic up to the one final
    conversion, so a flat patch has var = 0 EXACTLY (as in the naive two-pass loop) and everywhere else the two agree
    to the naive loop's own fp64 rounding.  (With fp64 tables the error was 1e-6 HU^2, i.e. a spurious sigma of
    1e-3 HU in flat air, enough to move the whole-schedule field of config 4 by 1e-2 voxel.)"""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(40, 36, 20))
    for v, R in ((ct, 3), (cbct, (4, 4, 1))):
        mean, var = oracle_mod.box_moments3(v, R)
        ms, vs = oracle_mod.box_moments3(v, R, sat=True)
        assert np.abs(ms - mean).max() < 1e-11
        assert np.abs(vs - var).max() < 1e-8 and (np.abs(vs - var) <= 1e-12 * var + 1e-13).all()
        assert vs.min() >= 0.0
        assert ((var == 0.0) == (vs == 0.0)).all() and (var == 0.0).any() == (v is ct)
    # values below 2^-7 HU are rounded to 2^-30 HU; values beyond +-16384 are refused (outputs left untouched)
    tiny = np.array([[[1e-3, 2e-3, -3e-3, 5e-4]]], dtype=np.float32)
    m1, v1 = oracle_mod.box_moments3(tiny, (1, 0, 0))
    m2, v2 = oracle_mod.box_moments3(tiny, (1, 0, 0), sat=True)
    assert np.abs(m1 - m2).max() < 1e-9 and np.abs(v1 - v2).max() < 1e-11


# ---------------------------------------------------------------- NEXT-4: pyramid with per-axis factors
def test_pyramid3(oracle_mod):
    rng = np.random.default_rng(4)
    v = rng.normal(size=(8, 12, 16)).astype(np.float32)
    r = rng.normal(size=(3, 4, 6, 8)).astype(np.float32)
    # all factors 2 = the hot path's operators, bit for bit
    assert np.array_equal(oracle_mod.downsample3(v, (2, 2, 2)), oracle_mod.downsample(v))
    assert np.array_equal(oracle_mod.upsample_field3(r, (2, 2, 2)), oracle_mod.upsample_field(r))
    # all factors 1 = identity
    assert np.array_equal(oracle_mod.downsample3(v, (1, 1, 1)), v)
    assert np.array_equal(oracle_mod.upsample_field3(r, (1, 1, 1)), r)
    # in-plane only: block mean over 2x2x1, written out
    d = oracle_mod.downsample3(v, (2, 2, 1))
    ref = v.astype(np.float64).reshape(8, 6, 2, 8, 2).mean(axis=(2, 4))
    assert d.shape == (8, 6, 8)
    np.testing.assert_allclose(d, ref, atol=1e-7)
    # up: z untouched (no mixing between slices, z component not doubled), x and y doubled at i/2 - 1/4
    up = oracle_mod.upsample_field3(r, (2, 2, 1))
    assert up.shape == (3, 4, 12, 16)
    const = np.ones((3, 4, 6, 8), dtype=np.float32) * np.array([1.0, 2.0, 3.0], dtype=np.float32)[:, None, None, None]
    upc = oracle_mod.upsample_field3(const, (2, 2, 1))
    assert np.all(upc[0] == 2.0) and np.all(upc[1] == 4.0) and np.all(upc[2] == 3.0)
    z, y, x = np.meshgrid(np.arange(4.0), np.arange(6.0), np.arange(8.0), indexing="ij")
    ramp = np.stack([0.5 * x + z, 0.25 * y, 2.0 * z]).astype(np.float32)
    upr = oracle_mod.upsample_field3(ramp, (2, 2, 1))
    zf, yf, xf = np.meshgrid(np.arange(4.0), np.arange(12.0), np.arange(16.0), indexing="ij")
    inner = (slice(None), slice(1, -1), slice(1, -1))
    np.testing.assert_allclose(upr[0][inner], (2 * (0.5 * (xf / 2 - 0.25) + zf))[inner], atol=1e-6)
    np.testing.assert_allclose(upr[1][inner], (2 * 0.25 * (yf / 2 - 0.25))[inner], atol=1e-6)
    np.testing.assert_allclose(upr[2][inner], (2.0 * zf)[inner], atol=1e-6)
    # each slice of the in-plane up-sampling equals the 2-D up-sampling of that slice alone
    one = oracle_mod.upsample_field3(r[:, 1:2], (2, 2, 1))
    assert np.array_equal(one[:, 0], up[:, 1])


# ---------------------------------------------------------------- NEXT-1: a, b, mask, interpolation
def test_ab_from_moments_matches_eq4(oracle_mod):
    """Eq. (4): with the voxel's own frozen (a, b), E(aS + b) = E(M) and E((aS + b)^2) = E(M^2)
    over the patch -- checked by explicit slicing; and a I_s + b is the hot path's a (I_s - mu_s) + mu_m."""
    rng = np.random.default_rng(6)
    s = rng.uniform(-200, 400, size=(6, 7, 8)).astype(np.float32)
    m = rng.uniform(-100, 900, size=(6, 7, 8)).astype(np.float32)
    R = 1
    mus, vs = oracle_mod.box_moments(s, R)
    mum, vm = oracle_mod.box_moments(m, R)
    a, b = oracle_mod.ab_from_moments(mus, vs, mum, vm)
    for z, y, x in [(0, 0, 0), (3, 3, 3), (5, 6, 7), (2, 0, 4)]:
        sl = (slice(max(z - R, 0), z + R + 1), slice(max(y - R, 0), y + R + 1), slice(max(x - R, 0), x + R + 1))
        S, M = s[sl].astype(np.float64), m[sl].astype(np.float64)
        Sp = a[z, y, x] * S + b[z, y, x]
        assert abs(Sp.mean() - M.mean()) < 1e-9
        assert abs((Sp ** 2).mean() - (M ** 2).mean()) < 1e-6
        assert abs(a[z, y, x] - M.std() / S.std()) < 1e-12
    np.testing.assert_allclose(oracle_mod.apply_ab(s, a, b), oracle_mod.correct(s, m, R), atol=2e-4)
    # var_s <= eps_var: a = 0, b = mu_m (reading A5)
    a0, b0 = oracle_mod.ab_from_moments(np.array([3.0]), np.array([0.0]), np.array([7.0]), np.array([2.0]))
    assert a0[0] == 0.0 and b0[0] == 7.0


def test_mask_eq7_by_hand(oracle_mod):
    """Eq. (7): xi = 1 where |I_m - I_s| > HU_0, or a < a_min, or a > a_max; strict inequalities."""
    m = np.array([[[100.0, 100.0, 100.0, 100.0, 100.0, 100.0]]], dtype=np.float32)
    s = np.array([[[100.0, 150.0, 151.0, 49.0, 100.0, 100.0]]], dtype=np.float32)
    a = np.array([[[1.0, 1.0, 1.0, 1.0, 0.49, 1.51]]])
    xi = oracle_mod.mask(m, s, a, hu0=50.0, a_min=0.5, a_max=1.5)
    assert xi.ravel().tolist() == [0, 0, 1, 1, 1, 1]
    a = np.array([[[0.5, 1.5, 1.0, 1.0, 1.0, 1.0]]])          # the bounds themselves are inside
    assert oracle_mod.mask(m, m, a, 50.0, 0.5, 1.5).ravel().tolist() == [0] * 6


def test_fill_two_intensity_toy_patch_by_hand(oracle_mod):
    """Eqs. (8)-(10) on a 3x1x1 row: the masked centre voxel of intensity s0 sees two available
    neighbours at intensities s0 + 10 and s0 - 30 with h = 20:  w = exp(-100/400), exp(-900/400)."""
    s = np.array([[[110.0, 100.0, 70.0]]], dtype=np.float32)
    a = np.array([[[2.0, 99.0, 4.0]]])
    b = np.array([[[-5.0, 99.0, 7.0]]])
    xi = np.array([[[0, 1, 0]]], dtype=np.uint8)
    fa, fb, left, passes = oracle_mod.fill_ab(s, xi, a, b, fill_radius=1, h=20.0)
    w1, w2 = math.exp(-100.0 / 400.0), math.exp(-900.0 / 400.0)
    assert abs(fa[0, 0, 1] - (w1 * 2.0 + w2 * 4.0) / (w1 + w2)) < 1e-12
    assert abs(fb[0, 0, 1] - (w1 * -5.0 + w2 * 7.0) / (w1 + w2)) < 1e-12
    assert left.sum() == 0 and passes == 1
    assert fa[0, 0, 0] == 2.0 and fa[0, 0, 2] == 4.0 and fb[0, 0, 0] == -5.0 and fb[0, 0, 2] == 7.0
    # h -> infinity: plain average; h -> 0: the neighbour of closest intensity
    fa, _, _, _ = oracle_mod.fill_ab(s, xi, a, b, 1, 1e9)
    assert abs(fa[0, 0, 1] - 3.0) < 1e-9
    fa, _, _, _ = oracle_mod.fill_ab(s, xi, a, b, 1, 1e-3)
    assert fa[0, 0, 1] == 2.0
    # intensity differences so large that exp(-D^2/h^2) underflows in fp64 still give the quotient of Eqs. (8)-(9)
    s2 = np.array([[[3000.0, -1000.0, 2990.0]]], dtype=np.float32)
    fa, _, left, _ = oracle_mod.fill_ab(s2, xi, a, b, 1, 5.0)
    assert left.sum() == 0 and np.isfinite(fa).all()
    w = math.exp(-((4000.0 ** 2) - (3990.0 ** 2)) / 25.0)     # relative weight of the farther neighbour
    assert abs(fa[0, 0, 1] - (w * 2.0 + 1.0 * 4.0) / (w + 1.0)) < 1e-12


def test_fill_passes_and_invariants(oracle_mod):
    rng = np.random.default_rng(8)
    shape = (9, 10, 11)
    s = rng.uniform(0, 100, size=shape).astype(np.float32)
    a = rng.uniform(0.5, 1.5, size=shape)
    b = rng.uniform(-50, 50, size=shape)
    # xi = 0 everywhere: nothing changes, no pass runs
    xi0 = np.zeros(shape, dtype=np.uint8)
    fa, fb, left, passes = oracle_mod.fill_ab(s, xi0, a, b, 1, 30.0)
    assert np.array_equal(fa, a) and np.array_equal(fb, b) and passes == 0 and left.sum() == 0
    # a masked 5x5x5 block, T of radius 1: the shell fills in pass 1, the 3x3x3 core in pass 2, the centre in pass 3
    xi = np.zeros(shape, dtype=np.uint8)
    xi[2:7, 2:7, 3:8] = 1
    for cap, expect_left in [(1, 27), (2, 1), (3, 0), (64, 0)]:
        fa, fb, left, passes = oracle_mod.fill_ab(s, xi, a, b, 1, 30.0, max_passes=cap)
        assert left.sum() == expect_left and passes == min(cap, 3)
        if expect_left:
            assert left[4, 4, 5] == 1 and fa[4, 4, 5] == 0.0 and fb[4, 4, 5] == 0.0    # "Initially a = b = 0 for xi = 1"
        # the values of xi = 0 voxels are never changed
        assert np.array_equal(fa[xi == 0], a[xi == 0]) and np.array_equal(fb[xi == 0], b[xi == 0])
        # a weighted average lies between the extremes of what it averages
        assert fa[xi == 1].max() <= a[xi == 0].max() + 1e-12 and fa[(xi == 1) & (left == 0)].min() >= a[xi == 0].min() - 1e-12
    # with T of radius 2 the same block needs 2 passes
    assert oracle_mod.fill_ab(s, xi, a, b, 2, 30.0)[3] == 2
    # a Jacobi pass: a voxel filled in pass 1 is NOT seen by its neighbours in pass 1 -- the first-pass value of a
    # shell voxel equals the hand-computed average over its xi = 0 neighbours only
    z, y, x = 2, 2, 3                                              # a corner of the block
    fa1 = oracle_mod.fill_ab(s, xi, a, b, 1, 30.0, max_passes=1)[0]
    num = den = 0.0
    nb = [(zz, yy, xx) for zz in range(z - 1, z + 2) for yy in range(y - 1, y + 2) for xx in range(x - 1, x + 2) if xi[zz, yy, xx] == 0]
    dmin = min((float(s[p]) - float(s[z, y, x])) ** 2 for p in nb)
    for p in nb:
        w = math.exp(-(((float(s[p]) - float(s[z, y, x])) ** 2) - dmin) / 900.0)
        num += w * a[p]; den += w
    assert abs(fa1[z, y, x] - num / den) < 1e-12
    # everything masked: nothing can be found, the loop ends, a = b = 0
    fa, fb, left, passes = oracle_mod.fill_ab(s, np.ones(shape, dtype=np.uint8), a, b, 1, 30.0)
    assert left.all() and not fa.any() and not fb.any() and passes == 1


def test_delta_hu_and_median(oracle_mod):
    ct = np.array([[[10.0, 20.0, 30.0, 40.0]]], dtype=np.float32)
    cb = np.array([[[0.0, 0.0, 10.0, 10.0]]], dtype=np.float32)
    assert oracle_mod.delta_hu(ct, cb) == 20.0
    a = np.array([5.0, 1.0, 3.0, 2.0, 4.0, 9.0])
    ones = np.ones(6)
    assert oracle_mod.median_a(a, ones, ones) == 3.0                             # lower median of 6 values
    assert oracle_mod.median_a(a[:5], ones[:5], ones[:5]) == 3.0
    vs = np.array([1.0, 1.0, 0.0, 1.0, 1.0, 1.0]); vm = np.array([1.0, 1.0, 1.0, 1.0, 1.0, 0.0])
    assert oracle_mod.median_a(a, vs, vm) == 2.0                                 # {5, 1, 2, 4} -> lower median 2
    assert oracle_mod.median_a(a, 0 * ones, ones) == 1.0                         # nothing qualifies


# ---------------------------------------------------------------- the general driver
def test_register_ex_is_the_documented_composition(oracle_mod):
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(32, 24, 16))
    R, sigma, iters = 2, 1.5, 3
    r0, c0 = oracle_mod.register(ct, cbct, R, sigma, 2, iters)
    o = oracle_mod.register_ex(ct, cbct, R, sigma, 2, iters)
    assert np.array_equal(o["disp"], r0) and np.array_equal(o["corr"], c0) and o["iters_run"].tolist() == [iters, iters]
    # summed-area moments in the middle iteration: same result to rounding
    o2 = oracle_mod.register_ex(ct, cbct, R, sigma, 2, iters, sat_between=True)
    assert np.abs(o2["disp"] - r0).max() < 1e-5
    # Fig. 9 (e), (f): mean a, mean b of the first coarse iteration, recomputed from the step functions
    ct1, cb1 = oracle_mod.downsample(ct), oracle_mod.downsample(cbct)
    mus, vs = oracle_mod.box_moments(cb1, R)
    mum, vm = oracle_mod.box_moments(ct1, R)                                     # r = 0: I_m^(0) = ct
    a, b = oracle_mod.ab_from_moments(mus, vs, mum, vm)
    assert abs(o["mean_a"][0, 0] - a.mean()) < 1e-12 and abs(o["mean_b"][0, 0] - b.mean()) < 1e-9
    assert np.isfinite(o["mean_a"]).all() and np.isfinite(o["mean_b"]).all()
    # stopping criterion and double force through the general driver = the dedicated entry points
    d1, run1, l1 = oracle_mod.register_stop(ct, cbct, R, sigma, 2, 14, stop_eps=1e-2, double_force=True)
    o3 = oracle_mod.register_ex(ct, cbct, R, sigma, 2, 14, stop_eps=1e-2, double_force=True, want_corr=False)
    assert np.array_equal(o3["disp"], d1) and o3["iters_run"].tolist() == run1.tolist()


def test_register_ex_anisotropic_composition(oracle_mod):
    """NEXT-4: patch 5x5x3 and an in-plane pyramid on a 32x24x10 volume = the stepwise composition."""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(32, 24, 10))
    R, fac, sigma, iters = (2, 2, 1), (2, 2, 1), 1.5, 2
    o = oracle_mod.register_ex(ct, cbct, R, sigma, 2, iters, fac=fac)
    ct1, cb1 = oracle_mod.downsample3(ct, fac), oracle_mod.downsample3(cbct, fac)
    assert ct1.shape == (10, 12, 16)
    rr = np.zeros((3,) + ct1.shape, dtype=np.float32)
    for _ in range(iters):
        m = oracle_mod.warp(ct1, rr); rr = oracle_mod.demons_step(m, oracle_mod.correct3(cb1, m, R), rr, sigma)
    rr = oracle_mod.upsample_field3(rr, fac)
    for _ in range(iters):
        m = oracle_mod.warp(ct, rr); rr = oracle_mod.demons_step(m, oracle_mod.correct3(cbct, m, R), rr, sigma)
    assert np.array_equal(o["disp"], rr)
    assert np.array_equal(o["corr"], oracle_mod.correct3(cbct, oracle_mod.warp(ct, rr), R))


def test_register_ex_mask_composition_and_limits(oracle_mod):
    """NEXT-1 through the driver: the global shift, HU_0 = 2 |Delta HU|, a_m = median(A) before the DIR (PAPER.md:161,
    :165) and one masked iteration recomputed from the step functions; with a mask that never fires the run equals
    the unmasked path up to the rounding of a I_s + b against a (I_s - mu_s) + mu_m."""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(32, 24, 16))
    R, sigma = 2, 1.5
    o = oracle_mod.register_ex(ct, cbct, R, sigma, 1, 1, mask=True, fill_radius=1, h=40.0)
    dhu = oracle_mod.delta_hu(ct, cbct)
    cb = (cbct.astype(np.float64) + dhu).astype(np.float32)                      # "globally adjust"
    mus, vs = oracle_mod.box_moments(cb, R)
    mum, vm = oracle_mod.box_moments(ct, R)
    a, b = oracle_mod.ab_from_moments(mus, vs, mum, vm)
    a_m = oracle_mod.median_a(a, vs, vm)
    info = o["info"]
    assert info["delta_hu"] == dhu and info["hu0"] == 2 * abs(dhu) and info["a_m"] == a_m
    assert info["a_min"] == 0.5 * a_m and info["a_max"] == 1.5 * a_m
    xi = oracle_mod.mask(ct, cb, a, info["hu0"], info["a_min"], info["a_max"])
    assert 0 < xi.mean() < 1
    fa, fb, left, _ = oracle_mod.fill_ab(cb, xi, a, b, 1, 40.0)
    sp = oracle_mod.apply_ab(cb, fa, fb)
    rr = oracle_mod.demons_step(ct, sp, np.zeros((3,) + ct.shape, dtype=np.float32), sigma)
    assert np.array_equal(o["disp"], rr)
    assert abs(o["mean_a"][0, 0] - fa.mean()) < 1e-12
    # a mask that never fires
    o_off = oracle_mod.register_ex(ct, cbct, R, sigma, 2, 4)
    o_on = oracle_mod.register_ex(ct, cbct, R, sigma, 2, 4, mask=True, hu0=1e30, a_range=(0.0, 1e30))
    assert np.abs(o_on["disp"] - o_off["disp"]).max() < 1e-4


@pytest.mark.parametrize("levels,auto", [(1, False), (2, True)])
def test_stepwise_mask_chain_is_register_ex(oracle_mod, levels, auto):
    """tests/next1_chain.py (Alg. A1 with the mask, one oracle call per step -- what the GPU parity test drives with the
    CUDA path's Eq. (7) decisions) is, with its own decisions, bit for bit oracle.register_ex(mask=True)"""
    import next1_chain
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(32, 24, 16))
    R, sigma, iters, rt, h = 2, 1.5, 5, 2, 60.0
    kw = {} if auto else dict(hu0=180.0, a_range=(0.5, 1.7))
    o = oracle_mod.register_ex(ct, cbct, R, sigma, levels, iters, mask=True, fill_radius=rt, h=h, **kw)
    seen = []
    c = next1_chain.run(oracle_mod, ct, cbct, R, sigma, levels, iters, rt, h, decide=lambda l, k, m, s, a0, xi: (seen.append((l, k, xi.mean())), xi)[1], **kw)
    assert np.array_equal(c["disp"], o["disp"]) and np.array_equal(c["corr"], o["corr"])
    assert c["params"] == (o["info"]["hu0"], o["info"]["a_min"], o["info"]["a_max"])
    assert [lk[:2] for lk in seen] == [(l, k) for l in range(levels - 1, -1, -1) for k in range(iters)] + [(0, iters)]
    assert 0.0 < min(f for _, _, f in seen) and max(f for _, _, f in seen) < 1.0     # the mask fires, and not everywhere
    # decisions matter: flipping them all gives another registration (so a test that overrides them does test something)
    c2 = next1_chain.run(oracle_mod, ct, cbct, R, sigma, levels, 2, rt, h, decide=lambda l, k, m, s, a0, xi: ~xi, **kw)
    c3 = next1_chain.run(oracle_mod, ct, cbct, R, sigma, levels, 2, rt, h, **kw)
    assert np.abs(c2["disp"] - c3["disp"]).max() > 1e-3


def test_mask_bounds_the_noise_free_case(oracle_mod):
    """Why the paper masks a: on a NOISE-FREE CBCT, flat regions have sigma_s ~ 0 and a = sigma_m /
    sigma_s explodes; the unmasked loop then drifts (DESIGN.md findings).  With Eq. (7) and the
    interpolation of a, b the same input registers with a bounded field and a lower image error."""
    ct, _, _, _ = phantoms.make_pair(1, dims=(48, 48, 24))
    u = np.zeros((3,) + ct.shape, dtype=np.float32); u[0] = 2.0; u[1] = -1.0
    cbct = (0.9 * phantoms.pullback(ct, u) - 60.0).astype(np.float32)            # gain + offset, no noise
    target = phantoms.pullback(ct, u)
    kw = dict(R=2, sigma=1.5, levels=1, iters=100)
    off = oracle_mod.register_ex(ct, cbct, **kw)
    on = oracle_mod.register_ex(ct, cbct, mask=True, fill_radius=2, h=50.0, hu0=100.0, **kw)
    body = target > -500
    rm = lambda r: float(np.sqrt(np.mean((oracle_mod.warp(ct, r) - target)[body] ** 2)))
    rmse0 = float(np.sqrt(np.mean((ct - target)[body] ** 2)))
    # measured: unmasked 195 -> 92 HU and still drifting (max |r| 6.3 after 40 iterations, 9.8 after 100);
    # masked 195 -> 40 HU, max |r| 3.8 for a true shift of (2, -1, 0)
    assert np.abs(on["disp"]).max() < 5.0 < np.abs(off["disp"]).max()
    assert rm(on["disp"]) < 0.3 * rmse0
    assert rm(on["disp"]) < 0.6 * rm(off["disp"])

"""SURVEY NEXT-1 on the CUDA path: a, b of Eqs. (5)-(6), the reliability mask of Eq. (7), the interpolation of
Eqs. (8)-(10), I'_s = a I_s + b, the global Delta-HU shift and the parameter rules HU_0 = 2 Delta HU, a_min/a_max =
0.5/1.5 median(A), and the Fig.-9 averages, against the oracle.

Eq. (7) is a threshold decision on floating-point values.  In the per-kernel tests both sides see the same fp32 inputs:
|I_m - I_s| > HU_0 is taken in fp64 on both (identical decisions); a is fp64 in the oracle and fp32 here, so a voxel whose
a lies within 1e-5 relative of a_min or a_max may fall on either side: the tests compare what is unique (everything away
from such voxels) and check that a disagreement, if any, sits exactly there.  In the whole loop the inputs of Eq. (7) are
chained results, and a voxel on the bound in some iteration is expected about once per run: the whole-loop test runs in
lock step with the oracle, checks that such a voxel does sit on a threshold, lets the oracle follow the CUDA path's
decision there, and then asserts the plain north_star bounds.
"""
import numpy as np
import pytest

import phantoms

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def disc():
    import __graft_entry__
    __graft_entry__.build()
    import paper_1204_6295_b200 as d
    assert torch.cuda.is_available()
    return d


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def get_ab(disc, ctx, shape, level=0):
    a, b = torch.empty(shape, device="cuda"), torch.empty(shape, device="cuda")
    xi = torch.empty(shape, device="cuda", dtype=torch.uint8)
    disc.disc_get_ab(ctx, level, a, b, xi)
    return a.cpu().numpy(), b.cpu().numpy(), xi.cpu().numpy()


def case(dims=(48, 40, 24)):
    ct, cbct, u, p = phantoms.make_pair(1, dims=dims)
    m = phantoms.pullback(ct, (0.5 * u).astype(np.float32)).astype(np.float32)     # a partly registered CT
    return ct, cbct, m


def test_ab_without_a_firing_mask(disc, oracle_mod):
    """Eqs. (5)-(6) and a I_s + b: with thresholds that never fire the masked path is the plain correction"""
    ct, cbct, m = case()
    R = 2
    nz, ny, nx = ct.shape
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, 1.5, 1, 1)
    disc.disc_set_mask(ctx, True, hu0=1e30, a_min=0.0, a_max=1e30, fill_radius=1, h=50.0)
    out = torch.empty(ct.shape, device="cuda")
    disc.disc_correct_intensity(ctx, 0, dev(cbct), dev(m), out)
    a, b, xi = get_ab(disc, ctx, ct.shape)
    mus, vs = oracle_mod.box_moments(cbct, R)
    mum, vm = oracle_mod.box_moments(m, R)
    a_ref, b_ref = oracle_mod.ab_from_moments(mus, vs, mum, vm)
    span = float(max(m.max(), cbct.max()) - min(m.min(), cbct.min()))
    assert not xi.any()
    assert np.abs(a - a_ref).max() <= 1e-5 * max(1.0, a_ref.max())
    assert np.abs(b - b_ref).max() <= 1e-4 * span
    assert np.abs(out.cpu().numpy() - oracle_mod.apply_ab(cbct, a_ref, b_ref)).max() <= 1e-4 * span
    assert np.abs(out.cpu().numpy() - oracle_mod.correct(cbct, m, R)).max() <= 1e-4 * span
    disc.disc_destroy(ctx)


@pytest.mark.parametrize("rt,h", [(1, 40.0), (2, 25.0), (3, 200.0)])
def test_mask_and_fill_against_the_oracle(disc, oracle_mod, rt, h):
    ct, cbct, m = case()
    R = 2
    nz, ny, nx = ct.shape
    hu0, a_min, a_max = 150.0, 0.55, 1.65
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, 1.5, 1, 1)
    disc.disc_set_mask(ctx, True, hu0=hu0, a_min=a_min, a_max=a_max, fill_radius=rt, h=h)
    out = torch.empty(ct.shape, device="cuda")
    disc.disc_correct_intensity(ctx, 0, dev(cbct), dev(m), out)
    a, b, xi = get_ab(disc, ctx, ct.shape)
    disc.disc_destroy(ctx)
    mus, vs = oracle_mod.box_moments(cbct, R)
    mum, vm = oracle_mod.box_moments(m, R)
    a0, b0 = oracle_mod.ab_from_moments(mus, vs, mum, vm)
    xi_ref = oracle_mod.mask(m, cbct, a0, hu0, a_min, a_max)
    assert 0.02 < xi_ref.mean() < 0.9
    # Eq. (7): identical decisions, except possibly where a sits on a bound
    flips = (xi != 0) != (xi_ref != 0)
    border = (np.abs(a0 - a_min) <= 1e-5 * a_min) | (np.abs(a0 - a_max) <= 1e-5 * a_max)
    assert not (flips & ~border).any()
    assert flips.sum() == 0, "seeded input: no voxel on a bound"
    fa, fb, left, passes = oracle_mod.fill_ab(cbct, xi_ref, a0, b0, rt, h)
    # the pass in which each voxel was filled is unique: compare the stamps through a one-pass-at-a-time oracle run
    stamp = np.where(xi_ref != 0, 255, 0).astype(np.uint8)
    for p in range(1, passes + 1):
        _, _, left_p, _ = oracle_mod.fill_ab(cbct, xi_ref, a0, b0, rt, h, max_passes=p)
        stamp[(stamp == 255) & (left_p == 0)] = p
    assert np.array_equal(xi, stamp)
    span = float(max(m.max(), cbct.max()) - min(m.min(), cbct.min()))
    assert np.abs(a - fa).max() <= 2e-5 * max(1.0, np.abs(fa).max())
    assert np.abs(b - fb).max() <= 1e-4 * span
    assert np.abs(out.cpu().numpy() - oracle_mod.apply_ab(cbct, fa, fb)).max() <= 1e-4 * span
    # the procedure does not change a, b where xi = 0
    free = xi_ref == 0
    assert np.abs(a[free] - a0[free]).max() <= 1e-5 * max(1.0, a0.max())


def test_fill_passes_stamps_and_cap(disc, oracle_mod):
    """a masked 5x5x5 block, T of radius 1: shell in pass 1, 3x3x3 core in pass 2, centre in pass 3 (PAPER.md:139:
    "for some voxels, the values of xi may be 1 for all voxels in their neighbor T"); a cap of 2 passes leaves the centre
    with a = b = 0 and stamp 255"""
    rng = np.random.default_rng(3)
    shape = (12, 16, 20)
    cbct = rng.uniform(-200, 300, size=shape).astype(np.float32)
    m = (1.1 * cbct + 20).astype(np.float32)
    m[3:8, 4:9, 6:11] += 500.0                                   # |I_m - I_s| > HU_0 only inside the block
    nz, ny, nx = shape
    for cap, centre_stamp in ((8, 3), (2, 255)):
        ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), 1, 1.0, 1, 1)
        disc.disc_set_mask(ctx, True, hu0=400.0, a_min=0.0, a_max=1e30, fill_radius=1, h=100.0, max_fill_passes=cap)
        out = torch.empty(shape, device="cuda")
        disc.disc_correct_intensity(ctx, 0, dev(cbct), dev(m), out)
        a, b, xi = get_ab(disc, ctx, shape)
        disc.disc_destroy(ctx)
        blk = xi[3:8, 4:9, 6:11]
        assert (xi != 0).sum() == 125 and (blk[1:4, 1:4, 1:4] >= 2).all() and (blk == 1).sum() == 125 - 27
        assert blk[2, 2, 2] == centre_stamp and (blk[1:4, 1:4, 1:4] == 2).sum() == 26
        if centre_stamp == 255:
            assert a[5, 6, 8] == 0.0 and b[5, 6, 8] == 0.0 and out.cpu().numpy()[5, 6, 8] == 0.0
        else:
            # a weighted average lies between the extremes of what it averages
            free = xi == 0
            assert a[~free].max() <= a[free].max() + 1e-6 and a[~free].min() >= a[free].min() - 1e-6


def test_mask_parameters_from_the_images(disc, oracle_mod):
    """Delta HU = mean(CT) - mean(CBCT), HU_0 = 2 |Delta HU|, a_m = median(A) before the DIR"""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(64, 48, 24))
    R = 2
    nz, ny, nx = ct.shape
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, 1.5, 1, 1)
    disc.disc_set_mask(ctx, True)
    dhu, hu0, a_m, a_min, a_max = disc.disc_mask_params(ctx, dev(ct), dev(cbct))
    d_ref = oracle_mod.delta_hu(ct, cbct)
    mus, vs = oracle_mod.box_moments(cbct, R)
    mum, vm = oracle_mod.box_moments(ct, R)
    a0, _ = oracle_mod.ab_from_moments(mus, vs, mum, vm)
    am_ref = oracle_mod.median_a(a0, vs, vm)
    assert abs(dhu - d_ref) <= 1e-5 * abs(d_ref) + 1e-4 and abs(hu0 - 2 * abs(d_ref)) <= 1e-4 * abs(d_ref) + 1e-4
    assert abs(a_m - am_ref) <= 2e-6 * am_ref
    assert a_min == np.float32(0.5) * np.float32(a_m) and a_max == np.float32(1.5) * np.float32(a_m)
    # given bounds are kept, the rest is still derived
    disc.disc_set_mask(ctx, True, hu0=123.0, a_min=0.25, a_max=4.0)
    p = disc.disc_mask_params(ctx, dev(ct), dev(cbct))
    assert p[1] == 123.0 and p[3] == 0.25 and p[4] == 4.0 and abs(p[0] - d_ref) <= 1e-5 * abs(d_ref) + 1e-4
    disc.disc_destroy(ctx)


# margins inside which an Eq. (7) decision may fall on either side: |I_m - I_s| within D_MARGIN HU of HU_0 (the fp32 warp
# here and the fp64 warp of the oracle differ by ~1e-4 HU, and the chained fields by <= 1e-4 voxel x the steepest CT
# gradient of a few hundred HU per voxel), a within A_MARGIN (relative) of a_min or a_max (fp32 against fp64 quotient)
D_MARGIN, A_MARGIN = 5e-2, 1e-4


@pytest.mark.parametrize("levels,auto", [(1, False), (2, True)])
def test_register_with_the_mask(disc, oracle_mod, levels, auto):
    """the whole loop of Alg. A1 including "globally adjust" and step 2, decision-exact:

    (1) the masked loop runs stepwise through the C-ABI (disc_warp -> disc_correct_intensity -> disc_get_ab ->
        disc_demons_step, pyramid through disc_downsample / disc_upsample_field) in lock step with the oracle's step
        functions (tests/next1_chain.py, pinned to oracle.register_ex on CPU).  In every iteration the xi of the CUDA
        path is compared with the oracle's Eq. (7) on the oracle's own chained inputs; a voxel where they differ must
        sit within D_MARGIN / A_MARGIN of a threshold, and the oracle goes on with the CUDA path's decision.  Then plain
        bounds: the field within north_star's 1e-2 voxel at the end of every level, EVERY corrected voxel within
        1e-4 x range (+ the field error times the steepest CT gradient);
    (2) disc_register -- the fused loop -- against that stepwise CUDA run: the same kernels on the same values."""
    import next1_chain
    ct, cbct, u, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    R, sigma, iters, rt, h = 2, 1.5, 12, 2, 60.0
    nz, ny, nx = ct.shape
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, levels, iters)
    d_ct, d_cb = dev(ct), dev(cbct)
    if auto:
        disc.disc_set_mask(ctx, True, fill_radius=rt, h=h)
        dhu, hu0, a_m, a_min, a_max = disc.disc_mask_params(ctx, d_ct, d_cb)       # PAPER.md:165, kept in the context
    else:
        hu0, a_min, a_max = 180.0, 0.5, 1.7
        disc.disc_set_mask(ctx, True, hu0=hu0, a_min=a_min, a_max=a_max, fill_radius=rt, h=h)
    # the derived parameters against the oracle's rules, then both sides decide with the SAME thresholds
    ref_params = next1_chain.run(oracle_mod, ct, cbct, R, sigma, 1, 0, rt, h,
                                 **({} if auto else dict(hu0=hu0, a_range=(a_min, a_max))))
    for got, want in zip((hu0, a_min, a_max), ref_params["params"]):
        assert abs(got - want) <= 1e-5 * abs(want)
    cb_shift = ref_params["cbct_shift"]                                            # fp32(cbct + Delta HU)
    span = float(max(ct.max(), cb_shift.max()) - min(ct.min(), cb_shift.min()))
    steep = max(float(np.abs(np.diff(ct.astype(np.float64), axis=a)).max()) for a in range(3))

    # ---- the stepwise CUDA run: state on the device, one C-ABI call per step
    g = {"ct": [d_ct], "cb": [dev(cb_shift)], "r": None, "flips": 0, "masked": [], "worst_sp": 0.0}
    for l in range(1, levels):
        for key in ("ct", "cb"):
            out = torch.empty(next1_chain.level_shape(ct.shape, l), device="cuda")
            disc.disc_downsample(ctx, l - 1, g[key][-1], out)
            g[key].append(out)

    def gpu_correct(l):
        shp = next1_chain.level_shape(ct.shape, l)
        m, sp = torch.empty(shp, device="cuda"), torch.empty(shp, device="cuda")
        disc.disc_warp(ctx, l, g["ct"][l], g["r"], m)
        disc.disc_correct_intensity(ctx, l, g["cb"][l], m, sp)
        _, _, xi = get_ab(disc, ctx, shp, l)
        return m, sp, xi != 0

    def decide(l, k, m_o, cb_o, a0, xi_o):
        shp = next1_chain.level_shape(ct.shape, l)
        if g["r"] is None:
            g["r"] = torch.zeros((3,) + shp, device="cuda")
        elif g["r"].shape[1:] != shp:
            fine = torch.empty((3,) + shp, device="cuda")
            disc.disc_upsample_field(ctx, l + 1, g["r"], fine)
            g["r"] = fine
        m, sp, xi_g = gpu_correct(l)
        g["sp"], g["m"] = sp, m
        if k < iters:
            disc.disc_demons_step(ctx, l, m, sp, g["r"])
        flips = xi_g != xi_o
        if flips.any():
            dd = np.abs(np.abs(m_o.astype(np.float64) - cb_o.astype(np.float64)) - hu0)[flips]
            da = np.minimum(np.abs(a0 - a_min) / a_min, np.abs(a0 - a_max) / a_max)[flips]
            assert ((dd <= D_MARGIN) | (da <= A_MARGIN)).all(), (l, k, dd, da)
            g["flips"] += int(flips.sum())
        g["masked"].append(float(xi_g.mean()))
        return xi_g

    def after_level(l, r_o):
        err = float(np.abs(g["r"].cpu().numpy() - r_o).max())
        assert err <= 1e-2, (l, err)
        g["err_r"] = err

    ref = next1_chain.run(oracle_mod, ct, cbct, R, sigma, levels, iters, rt, h, params=(hu0, a_min, a_max), decide=decide,
                          after_level=after_level)
    assert g["flips"] <= 10 and 0.01 < min(g["masked"]) and max(g["masked"]) < 0.95, (g["flips"], g["masked"])
    r_step, corr_step = g["r"].cpu().numpy(), g["sp"].cpu().numpy()
    assert np.abs(r_step - ref["disp"]).max() <= 1e-2                                  # north_star, plain max-abs
    assert np.abs(corr_step - ref["corr"]).max() <= 1e-4 * span + 2.0 * g["err_r"] * steep + 1e-3   # every voxel

    # ---- the fused loop: disc_register (shift, parameters, pyramid, iterations, final correction in one call)
    disc.disc_set_diagnostics(ctx, True)
    d_r, d_c = torch.empty((3,) + ct.shape, device="cuda"), torch.empty(ct.shape, device="cuda")
    disc.disc_register(ctx, d_ct, d_cb, d_r, d_c)
    mean_a, mean_b = disc.disc_get_diagnostics(ctx)
    disc.disc_destroy(ctx)
    assert np.abs(d_r.cpu().numpy() - r_step).max() <= 1e-5 and np.abs(d_c.cpu().numpy() - corr_step).max() <= 1e-5 * span
    assert np.abs(d_r.cpu().numpy() - ref["disp"]).max() <= 1e-2
    # Fig. 9 (e), (f) against the unassisted oracle run (averages over all voxels: a stray decision moves them by 1e-5)
    kw = {} if auto else dict(hu0=hu0, a_range=(a_min, a_max))
    o = oracle_mod.register_ex(ct, cbct, R, sigma, levels, iters, mask=True, fill_radius=rt, h=h, want_corr=False, **kw)
    np.testing.assert_allclose(np.array(mean_a).reshape(levels, iters), o["mean_a"], rtol=2e-3, atol=1e-4)
    np.testing.assert_allclose(np.array(mean_b).reshape(levels, iters), o["mean_b"], rtol=2e-3, atol=0.05)


def test_diagnostics_without_the_mask(disc, oracle_mod):
    """Fig. 9 (e), (f) on the hot path: the averages of a and b per iteration, and the field is unchanged by asking"""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    R, sigma, levels, iters = 2, 1.5, 2, 6
    nz, ny, nx = ct.shape
    ref = oracle_mod.register_ex(ct, cbct, R, sigma, levels, iters)
    fields = []
    for diag in (False, True):
        ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, levels, iters)
        disc.disc_set_diagnostics(ctx, diag)
        d_r = torch.empty((3,) + ct.shape, device="cuda")
        disc.disc_register(ctx, dev(ct), dev(cbct), d_r, None)
        fields.append(d_r.cpu().numpy())
        if diag:
            mean_a, mean_b = disc.disc_get_diagnostics(ctx)
        disc.disc_destroy(ctx)
    assert np.array_equal(fields[0], fields[1])
    assert np.abs(fields[1] - ref["disp"]).max() <= 1e-2
    np.testing.assert_allclose(np.array(mean_a).reshape(levels, iters), ref["mean_a"], rtol=1e-4)
    np.testing.assert_allclose(np.array(mean_b).reshape(levels, iters), ref["mean_b"], rtol=1e-4, atol=1e-2)


@pytest.mark.parametrize("use_mask", [True, False])
def test_early_stop_leaves_ab_and_diagnostics_of_the_last_iteration_run(disc, oracle_mod, use_mask):
    """stopping criterion together with the mask / the Fig.-9 diagnostics: once a level has stopped, the
    launches still enqueued for it must leave a, b, xi alone (they would otherwise re-read a, b as E(M), VAR(M)), and the
    diagnostic slots of iterations not run read NaN as in the oracle"""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    R, sigma, iters, eps, rt, h = 2, 1.5, 40, 0.12, 2, 60.0      # eps: both levels trip with a margin > 1e-3
    nz, ny, nx = ct.shape
    mkw = dict(hu0=180.0, a_min=0.5, a_max=1.7, fill_radius=rt, h=h)
    okw = dict(mask=True, hu0=180.0, a_range=(0.5, 1.7), fill_radius=rt, h=h) if use_mask else {}

    def run_gpu(levels, n_iters, stop):
        ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, levels, n_iters)
        if use_mask:
            disc.disc_set_mask(ctx, True, **mkw)
        disc.disc_set_diagnostics(ctx, True)
        if stop:
            disc.disc_set_stop(ctx, eps)
        d_r = torch.empty((3,) + ct.shape, device="cuda")
        disc.disc_register(ctx, dev(ct), dev(cbct), d_r, None)       # no final correction: a, b are the loop's
        run = disc.disc_iterations_run(ctx)
        ab = [get_ab(disc, ctx, tuple(s // 2 ** l for s in ct.shape), l) for l in range(levels)]
        ma, mb = disc.disc_get_diagnostics(ctx)
        disc.disc_destroy(ctx)
        return run, ab, np.array(ma).reshape(levels, n_iters), np.array(mb).reshape(levels, n_iters), d_r.cpu().numpy()

    # one level: the stopped run must leave exactly what a fixed schedule of the same length leaves
    run, ab, ma, mb, r = run_gpu(1, iters, True)
    ref = oracle_mod.register_ex(ct, cbct, R, sigma, 1, iters, stop_eps=eps, want_corr=False, **okw)
    assert 10 < run[0] < iters and run == list(ref["iters_run"])
    run2, ab2, ma2, mb2, r2 = run_gpu(1, run[0], False)
    assert np.array_equal(r, r2)
    for got, want in list(zip(ab[0], ab2[0]))[:3 if use_mask else 2]:           # xi is only written with the mask on
        assert np.isfinite(got).all() and np.array_equal(got, want)
    assert np.array_equal(ma[0, :run[0]], ma2[0]) and np.isnan(ma[0, run[0]:]).all() and np.isnan(mb[0, run[0]:]).all()
    np.testing.assert_allclose(ma, ref["mean_a"], rtol=2e-3, atol=1e-4)          # NaN where the oracle has NaN
    np.testing.assert_allclose(mb, ref["mean_b"], rtol=2e-3, atol=0.05)
    # two levels: the coarse level stops early and its a, b stay finite and sane; the averages follow the oracle
    run, ab, ma, mb, r = run_gpu(2, iters, True)
    ref = oracle_mod.register_ex(ct, cbct, R, sigma, 2, iters, stop_eps=eps, want_corr=False, **okw)
    assert run == list(ref["iters_run"]) and run[1] < iters
    a1, b1, xi1 = ab[1]
    assert np.isfinite(a1).all() and np.isfinite(b1).all() and a1.min() >= 0.0 and a1.max() < 50.0
    assert abs(float(a1.astype(np.float64).mean()) - ref["mean_a"][0, run[1] - 1]) <= 2e-3 * abs(ref["mean_a"][0, run[1] - 1]) + 1e-4
    np.testing.assert_allclose(ma, ref["mean_a"], rtol=2e-3, atol=1e-4)
    np.testing.assert_allclose(mb, ref["mean_b"], rtol=2e-3, atol=0.05)
    assert np.abs(r - ref["disp"]).max() <= (5e-2 if use_mask else 1e-2)

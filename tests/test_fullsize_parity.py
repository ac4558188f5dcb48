"""Parity at BASELINE.json's full size, in the launch configuration bench.py times: config 3 (256x256x128, R = 5,
sigma = 2.0) and the largest single level of config 4 (512x512x128, R = 7) through the same C-ABI calls.

Every kernel is compared with the naive oracle element by element on the WHOLE volume (the patch moments and the
correction too: ~3 s at config 3, ~25 s at config 4's finest level on the box's 16 cores), two whole iterations of
config 3's finest level likewise, and the whole 3 x 100 schedule of config 3 -- the workload bench.py times --
against oracle.register at north_star's 1e-2 voxel (~2 min of oracle time).  Config 4's 4 x 100 schedule is in
tests/test_zz_config4_schedule.py.
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


@pytest.fixture(scope="module")
def pair3():
    return phantoms.make_pair(3)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def sample_indices(shape, rng, n_random=300):
    """flat voxel indices: the 8 corners, edge / face points, the seams of 16-, 32- and 64-wide tiles, random points"""
    nz, ny, nx = shape
    pts = [(z, y, x) for z in (0, nz - 1) for y in (0, ny - 1) for x in (0, nx - 1)]
    for v in (15, 16, 31, 32, 63, 64):
        pts += [(min(v, nz - 1), min(v, ny - 1), min(v, nx - 1)), (nz // 2, min(v, ny - 1), nx - 1), (0, ny // 2, min(v, nx - 1)),
                (min(v, nz - 1), 0, nx // 2)]
    pts += list(zip(rng.integers(0, nz, n_random), rng.integers(0, ny, n_random), rng.integers(0, nx, n_random)))
    return np.array(sorted({(int(z) * ny + int(y)) * nx + int(x) for z, y, x in pts}), dtype=np.int64)


def hu_range(*vols):
    return float(max(v.max() for v in vols) - min(v.min() for v in vols))


def test_config3_per_kernel_full_volume(disc, oracle_mod, pair3):
    ct, cbct, u, p = pair3
    nz, ny, nx = ct.shape
    R, sigma = p["patch_radius"], p["sigma"]
    rng = np.random.default_rng(7)
    r0 = (0.6 * u).astype(np.float32)
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, p["levels"], p["iters"])
    d_ct, d_cb, d_r0 = dev(ct), dev(cbct), dev(r0)
    span = hu_range(ct, cbct)
    # warp: whole volume
    d_m = torch.empty_like(d_ct)
    disc.disc_warp(ctx, 0, d_ct, d_r0, d_m)
    m = d_m.cpu().numpy()
    assert np.abs(m - oracle_mod.warp(ct, r0)).max() <= 1e-4 * span
    # correction and moments: EVERY voxel against the naive patch loops (PAPER.md:95 Eq. 3, :117-119 Eqs. 5-6)
    d_sp = torch.empty_like(d_ct)
    disc.disc_correct_intensity(ctx, 0, d_cb, d_m, d_sp)
    sp = d_sp.cpu().numpy()
    mu_s, var_s = oracle_mod.box_moments(cbct, R)
    mu_m, var_m = oracle_mod.box_moments(m, R)
    assert np.abs(sp - oracle_mod.correct_from_moments(cbct, mu_s, var_s, mu_m, var_m)).max() <= 1e-4 * span
    d_mu, d_var = torch.empty_like(d_ct), torch.empty_like(d_ct)
    disc.disc_box_moments(ctx, 0, d_cb, d_mu, d_var)
    assert np.abs(d_mu.cpu().numpy() - mu_s).max() <= 1e-4 * span
    assert np.abs(np.sqrt(d_var.cpu().numpy()) - np.sqrt(var_s)).max() <= 1e-4 * span
    # the sampler agrees with the whole-volume loop at the seams (it is pinned on CPU, tests/test_oracle_pins_ext.py)
    idx = sample_indices(ct.shape, rng, 50)
    assert np.array_equal(oracle_mod.box_moments_at(cbct, R, idx)[0], mu_s.ravel()[idx])
    # force + update, Gaussian, demons step: whole volume (same fp32 inputs on both sides)
    d_r = d_r0.clone()
    disc.disc_force_update(ctx, 0, d_m, d_sp, d_r)
    assert np.abs(d_r.cpu().numpy() - oracle_mod.force_update(m, sp, r0)).max() <= 1e-4
    d_r = d_r0.clone()
    disc.disc_smooth_field(ctx, 0, d_r)
    assert np.abs(d_r.cpu().numpy() - oracle_mod.smooth_field(r0, sigma)).max() <= 1e-4
    d_r = d_r0.clone()
    disc.disc_demons_step(ctx, 0, d_m, d_sp, d_r)
    assert np.abs(d_r.cpu().numpy() - oracle_mod.demons_step(m, sp, r0, sigma)).max() <= 1e-4
    disc.disc_destroy(ctx)


def test_config3_two_whole_iterations(disc, oracle_mod, pair3):
    """the fused per-iteration kernels (correct -> force+Gxy -> Gz+warp), 256x256x128, against the stepwise oracle"""
    ct, cbct, u, p = pair3
    nz, ny, nx = ct.shape
    R, sigma = p["patch_radius"], p["sigma"]
    r0 = (0.6 * u).astype(np.float32)
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, 1, 2)
    d_r = dev(r0)
    disc.disc_iterate(ctx, 0, dev(ct), dev(cbct), d_r, 2)
    rr = r0.copy()
    for _ in range(2):
        m = oracle_mod.warp(ct, rr)
        rr = oracle_mod.demons_step(m, oracle_mod.correct(cbct, m, R), rr, sigma)
    err = np.abs(d_r.cpu().numpy() - rr).max()
    disc.disc_destroy(ctx)
    assert err <= 1e-3, err


@pytest.mark.slow
def test_config3_whole_schedule_against_the_oracle(disc, oracle_mod, pair3):
    """north_star: "final displacement within 1e-2 voxel max-abs after the full schedule" on the benchmarked workload:
    256x256x128, 3 levels x 100 iterations, R = 5, sigma = 2 (Alg. A1), disc_register against
    oracle.register (naive patch loops throughout, ~2 min on 16 cores)."""
    ct, cbct, u, p = pair3
    nz, ny, nx = ct.shape
    R, sigma = p["patch_radius"], p["sigma"]
    assert (nx, ny, nz, R, p["levels"], p["iters"]) == (256, 256, 128, 5, 3, 100)
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, p["levels"], p["iters"])
    d_ct, d_cb = dev(ct), dev(cbct)
    d_r, d_corr = torch.empty((3,) + ct.shape, device="cuda"), torch.empty_like(d_ct)
    disc.disc_register(ctx, d_ct, d_cb, d_r, d_corr)
    # reading A12: the returned corrected CBCT is correct(cbct, warp(ct, out_disp)) -- the same kernels, so bit-exact
    d_m, d_c2 = torch.empty_like(d_ct), torch.empty_like(d_ct)
    disc.disc_warp(ctx, 0, d_ct, d_r, d_m)
    disc.disc_correct_intensity(ctx, 0, d_cb, d_m, d_c2)
    assert torch.equal(d_c2, d_corr)
    r, corr, m = d_r.cpu().numpy(), d_corr.cpu().numpy(), d_m.cpu().numpy()
    assert np.isfinite(r).all()
    r_ref, corr_ref = oracle_mod.register(ct, cbct, R, sigma, p["levels"], p["iters"])
    err_r = float(np.abs(r - r_ref).max())
    assert err_r <= 1e-2, f"field error {err_r} voxel after the 3 x 100 schedule"
    span = hu_range(ct, cbct)
    g = float(np.abs(np.stack(np.gradient(ct.astype(np.float64)))).max())
    err_c = float(np.abs(corr - corr_ref).max())
    assert err_c <= 1e-4 * span + 2.0 * err_r * g + 1e-3, (err_c, err_r, g)
    # the registration did its job: the deformed CT is closer to the deformation-only target ct(x + u) than the CT
    target = phantoms.pullback(ct, u)
    body = target > -500.0
    rmse0 = np.sqrt(np.mean((ct - target)[body] ** 2))
    rmse1 = np.sqrt(np.mean((m - target)[body] ** 2))
    assert rmse1 < 0.6 * rmse0, (rmse0, rmse1)
    # P10 (AM-GM): one more force update moves no component by more than 1/2 voxel
    d_r2 = d_r.clone()
    disc.disc_force_update(ctx, 0, d_m, d_corr, d_r2)
    assert float((d_r2 - d_r).abs().max()) <= 0.5 + 1e-6
    disc.disc_destroy(ctx)


@pytest.mark.slow
def test_config4_finest_level_whole_volume(disc, oracle_mod):
    """512x512x128, R = 7 (patch 15^3), K = 6: every kernel on the whole volume against the naive oracle"""
    dims, R, sigma = (512, 512, 128), 7, 2.0
    a, b, u = phantoms.make_sweep_inputs(dims, seed_offset=4)
    a = (a * 4.0).astype(np.float32)
    b = (0.9 * b * 4.0 - 100.0).astype(np.float32)
    nz, ny, nx = a.shape
    ctx = disc.disc_create(dims, (1, 1, 1), R, sigma, 4, 1)
    span = hu_range(a, b)
    d_a, d_b, d_u = dev(a), dev(b), dev(u)
    d_sp = torch.empty_like(d_a)
    disc.disc_correct_intensity(ctx, 0, d_b, d_a, d_sp)
    sp = d_sp.cpu().numpy()
    mu_s, var_s = oracle_mod.box_moments(b, R)
    mu_m, var_m = oracle_mod.box_moments(a, R)
    assert np.abs(sp - oracle_mod.correct_from_moments(b, mu_s, var_s, mu_m, var_m)).max() <= 1e-4 * span
    d_mu, d_var = torch.empty_like(d_a), torch.empty_like(d_a)
    disc.disc_box_moments(ctx, 0, d_b, d_mu, d_var)
    assert np.abs(d_mu.cpu().numpy() - mu_s).max() <= 1e-4 * span
    assert np.abs(np.sqrt(d_var.cpu().numpy()) - np.sqrt(var_s)).max() <= 1e-4 * span
    del mu_s, var_s, mu_m, var_m, d_mu, d_var
    d_r = d_u.clone()
    disc.disc_demons_step(ctx, 0, d_a, d_sp, d_r)
    assert np.abs(d_r.cpu().numpy() - oracle_mod.demons_step(a, sp, u, sigma)).max() <= 1e-4
    d_m = torch.empty_like(d_a)
    disc.disc_warp(ctx, 0, d_a, d_u, d_m)
    assert np.abs(d_m.cpu().numpy() - oracle_mod.warp(a, u)).max() <= 1e-4 * span
    disc.disc_destroy(ctx)

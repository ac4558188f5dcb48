"""Whole-schedule parity: disc_register / disc_iterate on the GPU against oracle.register on the same seeded
phantoms.  Tolerance (north_star): final displacement max-abs <= 1e-2 voxel after the full schedule; corrected
CBCT max-abs <= 1e-4 x intensity range (plus the field tolerance times the steepest edge, because the corrected
image is evaluated at the GPU's own final field)."""
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


def gpu_register(disc, ct, cbct, R, sigma, levels, iters, host=False, double_force=False):
    nz, ny, nx = ct.shape
    ctx = disc.disc_create((nx, ny, nz), (1.0, 1.0, 1.0), R, sigma, levels, iters)
    if double_force:
        disc.disc_set_force(ctx, disc.DISC_FORCE_DOUBLE)
    if host:
        r = np.empty((3,) + ct.shape, dtype=np.float32)
        corr = np.empty_like(ct)
        disc.disc_register_host(ctx, ct, cbct, r, corr)
    else:
        d_r = torch.empty((3,) + ct.shape, device="cuda")
        d_c = torch.empty(ct.shape, device="cuda")
        disc.disc_register(ctx, dev(ct), dev(cbct), d_r, d_c)
        torch.cuda.synchronize()
        r, corr = d_r.cpu().numpy(), d_c.cpu().numpy()
    n = disc.disc_launch_count(ctx)
    disc.disc_destroy(ctx)
    return r, corr, n


def check(ct, cbct, r, corr, r_ref, corr_ref):
    err_r = np.abs(r - r_ref).max()
    assert err_r <= 1e-2, f"field error {err_r} voxel"
    rng = float(max(ct.max(), cbct.max()) - min(ct.min(), cbct.min()))
    g = np.abs(np.stack(np.gradient(ct.astype(np.float64)))).max()
    err_c = np.abs(corr - corr_ref).max()
    assert err_c <= 1e-4 * rng + 2.0 * err_r * g + 1e-3, f"corrected cbct error {err_c} HU (field err {err_r}, grad {g})"
    return err_r, err_c


@pytest.mark.parametrize("dims,R,sigma,levels,iters", [
    ((24, 20, 12), 1, 1.0, 1, 5),
    ((40, 36, 20), 2, 1.5, 2, 10),
    ((70, 44, 24), 3, 2.0, 3, 8),        # ragged tiles at every level
    ((32, 32, 16), 0, 1.5, 1, 4),        # R = 0: s' = m, no force
])
def test_register_small(disc, oracle_mod, dims, R, sigma, levels, iters):
    dims = tuple(d - d % (1 << (levels - 1)) for d in dims)
    ct, cbct, _, _ = phantoms.make_pair(1, dims=dims)
    r, corr, n = gpu_register(disc, ct, cbct, R, sigma, levels, iters)
    r_ref, corr_ref = oracle_mod.register(ct, cbct, R, sigma, levels, iters)
    check(ct, cbct, r, corr, r_ref, corr_ref)
    assert n >= 3 * levels * iters


def test_register_config1_full_schedule(disc, oracle_mod):
    ct, cbct, u, p = phantoms.make_pair(1)
    args = (p["patch_radius"], p["sigma"], p["levels"], p["iters"])
    r, corr, _ = gpu_register(disc, ct, cbct, *args)
    r_ref, corr_ref = oracle_mod.register(ct, cbct, *args)
    err_r, err_c = check(ct, cbct, r, corr, r_ref, corr_ref)
    print(f"config 1: max|dr| = {err_r:.2e} voxel, max|dcorr| = {err_c:.2e} HU")
    # the host-buffer entry point gives the same answer
    r2, corr2, _ = gpu_register(disc, ct, cbct, *args, host=True)
    assert np.array_equal(r2, r) and np.array_equal(corr2, corr)


@pytest.mark.slow
def test_register_config2_full_schedule(disc, oracle_mod):
    ct, cbct, u, p = phantoms.make_pair(2)
    args = (p["patch_radius"], p["sigma"], p["levels"], p["iters"])
    r, corr, _ = gpu_register(disc, ct, cbct, *args)
    r_ref, corr_ref = oracle_mod.register(ct, cbct, *args)
    err_r, err_c = check(ct, cbct, r, corr, r_ref, corr_ref)
    print(f"config 2: max|dr| = {err_r:.2e} voxel, max|dcorr| = {err_c:.2e} HU")


def test_iterate_matches_stepwise_oracle(disc, oracle_mod):
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    R, sigma, n_it = 2, 1.5, 6
    r0 = (0.5 * phantoms.disp_smooth_random((48, 40, 24), np.random.default_rng(3), max_disp=2.0)).astype(np.float32)
    ctx = disc.disc_create((48, 40, 24), (1, 1, 1), R, sigma, 1, n_it)
    d_r = dev(r0)
    disc.disc_iterate(ctx, 0, dev(ct), dev(cbct), d_r, n_it)
    rr = r0.copy()
    for _ in range(n_it):
        m = oracle_mod.warp(ct, rr)
        rr = oracle_mod.demons_step(m, oracle_mod.correct(cbct, m, R), rr, sigma)
    assert np.abs(d_r.cpu().numpy() - rr).max() <= 1e-3


@pytest.mark.parametrize("dims,R,sigma,levels,iters", [
    ((40, 36, 20), 2, 1.5, 2, 10),
    ((64, 64, 32), 3, 1.5, 1, 50),       # config 1's schedule
    ((70, 44, 24), 3, 2.0, 3, 8),
])
def test_register_double_force(disc, oracle_mod, dims, R, sigma, levels, iters):
    """the whole schedule with both terms of Eq. (1)"""
    dims = tuple(d - d % (1 << (levels - 1)) for d in dims)
    ct, cbct, _, _ = phantoms.make_pair(1, dims=dims)
    r, corr, _ = gpu_register(disc, ct, cbct, R, sigma, levels, iters, double_force=True)
    r_ref, corr_ref = oracle_mod.register(ct, cbct, R, sigma, levels, iters, double_force=True)
    check(ct, cbct, r, corr, r_ref, corr_ref)
    r1, _ = oracle_mod.register(ct, cbct, R, sigma, levels, iters, want_corr=False)
    assert np.abs(r_ref - r1).max() > 0.05      # and it is a different registration than the Thirion one


@pytest.mark.parametrize("dims,R,sigma,levels,iters,eps,double_force", [
    ((48, 40, 24), 3, 1.5, 2, 40, 2e-3, False),
    ((64, 64, 32), 3, 1.5, 1, 50, 4e-2, False),      # config 1's schedule with the criterion on (trips at k = 32)
    ((48, 40, 24), 2, 2.0, 2, 30, 5e-3, True),
    ((40, 36, 20), 2, 1.5, 2, 14, 1e-4, False),      # the paper's eps: nothing trips, all iterations run
    ((44, 40, 24), 2, 1.5, 2, 30, 3e-3, False),      # nx = 22 at the coarse level: the plain-load force kernel, whose
                                                     # sums come from the separate k_force_norms launch
])
def test_register_stopping_criterion(disc, oracle_mod, dims, R, sigma, levels, iters, eps, double_force):
    """NEXT-3: the device-side criterion stops each level where the oracle's does.  The decision
    compares two floating-point ratios with eps; where the oracle's own margin to eps is below 1e-6 either count is
    correct, and the field is then checked against the oracle run with the GPU's counts."""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=dims)
    nz, ny, nx = ct.shape
    ctx = disc.disc_create((nx, ny, nz), (1.0, 1.0, 1.0), R, sigma, levels, iters)
    if double_force:
        disc.disc_set_force(ctx, disc.DISC_FORCE_DOUBLE)
    disc.disc_set_stop(ctx, eps)
    d_r = torch.empty((3,) + ct.shape, device="cuda")
    d_c = torch.empty(ct.shape, device="cuda")
    disc.disc_register(ctx, dev(ct), dev(cbct), d_r, d_c)
    run = np.array(disc.disc_iterations_run(ctx))
    r_ref, run_ref, lt = oracle_mod.register_stop(ct, cbct, R, sigma, levels, iters, stop_eps=eps, double_force=double_force)
    if not np.array_equal(run, run_ref):
        for lev in range(levels):
            if run[lev] != run_ref[lev]:
                k = min(run[lev], run_ref[lev]) - 1            # the iteration where the two decisions differ
                row = lt[levels - 1 - lev]
                assert k >= 10 and abs(row[k - 10] - row[k] - eps) < 1e-6, (lev, run, run_ref)
                break                                           # later levels start from different fields
        r_ref, _, _ = oracle_mod.register_stop(ct, cbct, R, sigma, levels, iters, iters_per_level=run, double_force=double_force)
    assert np.abs(d_r.cpu().numpy() - r_ref).max() <= 1e-2
    if eps > 1e-4:
        assert run.min() < iters                                # the case is meant to stop early somewhere
    else:
        assert np.all(run == iters)
    # reading A12 still holds after an early stop: the returned corrected CBCT belongs to the returned field
    d_m, d_c2 = torch.empty_like(d_c), torch.empty_like(d_c)
    disc.disc_warp(ctx, 0, dev(ct), d_r, d_m)
    disc.disc_correct_intensity(ctx, 0, dev(cbct), d_m, d_c2)
    assert torch.equal(d_c2, d_c)
    # switching the criterion off restores the fixed schedule
    disc.disc_set_stop(ctx, -1.0)
    disc.disc_register(ctx, dev(ct), dev(cbct), d_r, d_c)
    assert disc.disc_iterations_run(ctx) == [iters] * levels
    r_fix, _ = oracle_mod.register(ct, cbct, R, sigma, levels, iters, want_corr=False, double_force=double_force)
    assert np.abs(d_r.cpu().numpy() - r_fix).max() <= 1e-2
    disc.disc_destroy(ctx)


def test_register_degenerate_schedules(disc, oracle_mod):
    """edge cases of the driver: zero iterations (the field stays zero, the corrected CBCT is correct(cbct, ct)), a
    one-voxel-thick volume, and a volume with a single column"""
    ct, cbct, _, _ = phantoms.make_pair(1, dims=(32, 24, 16))
    r, corr, n = gpu_register(disc, ct, cbct, 2, 1.5, 2, 0)
    assert not r.any()
    span = float(max(ct.max(), cbct.max()) - min(ct.min(), cbct.min()))
    assert np.abs(corr - oracle_mod.correct(cbct, ct, 2)).max() <= 1e-4 * span
    for dims in ((20, 18, 1), (1, 1, 24), (4, 1, 6)):
        ct2, cbct2, _, _ = phantoms.make_pair(1, dims=dims)
        r, corr, _ = gpu_register(disc, ct2, cbct2, 1, 1.0, 1, 6)
        r_ref, corr_ref = oracle_mod.register(ct2, cbct2, 1, 1.0, 1, 6)
        err_r = np.abs(r - r_ref).max()
        assert err_r <= 1e-2, (dims, err_r)
        span = float(max(ct2.max(), cbct2.max()) - min(ct2.min(), cbct2.min()))
        steep = max([np.abs(np.diff(ct2.astype(np.float64), axis=a)).max() for a in range(3) if ct2.shape[a] > 1] + [0.0])
        assert np.abs(corr - corr_ref).max() <= 1e-4 * span + 2.0 * err_r * steep + 1e-3, dims

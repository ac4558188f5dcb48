"""Parity at the sizes of BASELINE.json's config 5 that no other test reaches -- 256^3 and 512x512x256 -- for each kernel
the per-kernel sweep (bench.py --sweep) times, on the sweep's own seeded inputs and through the same C-ABI calls in the
same launch configuration (one-level context, the sweep's radii and sigmas).

warp, force + update and the Gaussian are compared with the oracle on the WHOLE volume; the patch moments (whose naive
loops cost n = (2R+1)^3 per voxel) on sampled voxels through the oracle's `_at` samplers (pinned on CPU against the
whole-volume loops): the 8 corners, face and edge points, the seams of 16-, 32- and 64-wide tiles and of the z chunks,
and random interior points.  Tolerances as in tests/test_kernels_parity.py.
"""
import numpy as np
import pytest

import phantoms

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

torch = pytest.importorskip("torch")

SIZES = [(256, 256, 256), (512, 512, 256)]


@pytest.fixture(scope="module")
def disc():
    import __graft_entry__
    __graft_entry__.build()
    import paper_1204_6295_b200 as d
    assert torch.cuda.is_available()
    return d


@pytest.fixture(scope="module", params=SIZES, ids=lambda d: "x".join(map(str, d)))
def inputs(request):
    dims = request.param
    a, b, u = phantoms.make_sweep_inputs(dims)
    return dims, a, b, u


def sample_indices(shape, rng, n_random):
    nz, ny, nx = shape
    pts = [(z, y, x) for z in (0, nz - 1) for y in (0, ny - 1) for x in (0, nx - 1)]
    for v in (15, 16, 31, 32, 63, 64, 127, 128):
        pts += [(min(v, nz - 1), min(v, ny - 1), min(v, nx - 1)), (nz // 2, min(v, ny - 1), nx - 1), (0, ny // 2, min(v, nx - 1)),
                (min(v, nz - 1), 0, nx // 2), (min(v, nz - 1), ny // 3, nx // 3)]
    pts += list(zip(rng.integers(0, nz, n_random), rng.integers(0, ny, n_random), rng.integers(0, nx, n_random)))
    return np.array(sorted({(int(z) * ny + int(y)) * nx + int(x) for z, y, x in pts}), dtype=np.int64)


def test_warp_and_force_whole_volume(disc, oracle_mod, inputs):
    dims, a, b, u = inputs
    span = float(max(a.max(), b.max()) - min(a.min(), b.min()))
    ctx = disc.disc_create(dims, (1.0, 1.0, 1.0), 1, 1.0, 1, 1)
    d_a, d_u = torch.from_numpy(a).cuda(), torch.from_numpy(u).cuda()
    d_o = torch.empty_like(d_a)
    disc.disc_warp(ctx, 0, d_a, d_u, d_o)
    got = d_o.cpu().numpy()
    del d_o
    assert np.abs(got - oracle_mod.warp(a, u)).max() <= 1e-4 * span
    d_b = torch.from_numpy(b).cuda()
    disc.disc_force_update(ctx, 0, d_a, d_b, d_u)
    got = d_u.cpu().numpy()
    disc.disc_destroy(ctx)
    del d_a, d_b, d_u
    torch.cuda.empty_cache()
    assert np.abs(got - oracle_mod.force_update(a, b, u)).max() <= 1e-4


@pytest.mark.parametrize("sigma", [1.0, 2.0, 3.0])
def test_smooth_field_whole_volume(disc, oracle_mod, inputs, sigma):
    dims, a, b, u = inputs
    ctx = disc.disc_create(dims, (1.0, 1.0, 1.0), 1, sigma, 1, 1)
    d_u = torch.from_numpy(u).cuda()
    disc.disc_smooth_field(ctx, 0, d_u)
    got = d_u.cpu().numpy()
    disc.disc_destroy(ctx)
    del d_u
    torch.cuda.empty_cache()
    assert np.abs(got - oracle_mod.smooth_field(u, sigma)).max() <= 1e-4


@pytest.mark.parametrize("R", [1, 5, 8, 10])
def test_box_moments_sampled(disc, oracle_mod, inputs, R):
    dims, a, b, u = inputs
    span = float(a.max() - a.min())
    ctx = disc.disc_create(dims, (1.0, 1.0, 1.0), R, 1.0, 1, 1)
    d_a = torch.from_numpy(a).cuda()
    d_mu, d_var = torch.empty_like(d_a), torch.empty_like(d_a)
    disc.disc_box_moments(ctx, 0, d_a, d_mu, d_var)
    idx = sample_indices(a.shape, np.random.default_rng(70 + R), 3000 if R <= 5 else 1200)
    t_idx = torch.from_numpy(idx).cuda()
    mu, var = d_mu.flatten()[t_idx].cpu().numpy(), d_var.flatten()[t_idx].cpu().numpy()
    assert torch.isfinite(d_mu).all() and torch.isfinite(d_var).all() and (d_var >= 0).all()
    # correction through the same kernels (z-score of a, then sigma_m zhat + mu_m with m = b)
    d_b, d_c = torch.from_numpy(b).cuda(), torch.empty_like(d_a)
    disc.disc_correct_intensity(ctx, 0, d_a, d_b, d_c)
    corr = d_c.flatten()[t_idx].cpu().numpy()
    disc.disc_destroy(ctx)
    del d_a, d_b, d_c, d_mu, d_var
    torch.cuda.empty_cache()
    mu_ref, var_ref = oracle_mod.box_moments_at(a, R, idx)
    assert np.abs(mu - mu_ref).max() <= 1e-4 * span
    assert np.abs(np.sqrt(var) - np.sqrt(var_ref)).max() <= 1e-4 * span
    span2 = float(max(a.max(), b.max()) - min(a.min(), b.min()))
    assert np.abs(corr - oracle_mod.correct_at(a, b, R, idx)).max() <= 1e-4 * span2

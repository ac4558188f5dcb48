"""SURVEY NEXT-4 on the CUDA path: non-cubic patches (3x3x3 ... 25x25x7), a pyramid that halves only the
transverse plane and a slice count that no power of two divides (256x256x68 at 0.94x0.94x2.5 mm), through
disc_create_ex, against the oracle's per-axis functions.  Same tolerances as the cubic path.
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


def rand_pair(shape, seed):
    rng = np.random.default_rng(seed)
    m = rng.uniform(-1000, 1500, size=shape).astype(np.float32)
    s = (0.8 * m + rng.normal(0, 60, size=shape) - 50).astype(np.float32)
    return m, s


# shapes [nz, ny, nx]: nx % 4 == 0 takes the TMA kernel, the others the plain-definition fallback
@pytest.mark.parametrize("shape", [(13, 40, 72), (20, 70, 36), (9, 21, 35), (6, 33, 64)])
@pytest.mark.parametrize("R", [(1, 1, 1), (2, 2, 1), (5, 5, 1), (12, 12, 3), (3, 3, 0), (0, 0, 2), (4, 4, 7), (2, 2, 9)])
def test_moments_and_correction_anisotropic(disc, oracle_mod, shape, R):
    nz, ny, nx = shape
    m, s = rand_pair(shape, 7 + sum(R))
    ctx = disc.disc_create_ex((nx, ny, nz), (0.94, 0.94, 2.5), R, 1.5, 1, 1, (2, 2, 1))
    span = float(max(m.max(), s.max()) - min(m.min(), s.min()))
    mu, var = torch.empty(shape, device="cuda"), torch.empty(shape, device="cuda")
    disc.disc_box_moments(ctx, 0, dev(s), mu, var)
    mu_ref, var_ref = oracle_mod.box_moments3(s, R)
    assert np.abs(mu.cpu().numpy() - mu_ref).max() <= 1e-4 * span
    assert np.abs(np.sqrt(var.cpu().numpy()) - np.sqrt(var_ref)).max() <= 1e-4 * span
    out = torch.empty(shape, device="cuda")
    disc.disc_correct_intensity(ctx, 0, dev(s), dev(m), out)
    assert np.abs(out.cpu().numpy() - oracle_mod.correct3(s, m, R)).max() <= 1e-4 * span
    disc.disc_destroy(ctx)


def test_anisotropic_ramp_variance_closed_form(disc):
    """sum_c g_c^2 R_c (R_c + 1) / 3 in the interior of a linear ramp, on the CUDA path itself (patch 25x25x7)"""
    R, g = (12, 12, 3), (1.5, -2.0, 0.25)
    nx, ny, nz = 64, 40, 12
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    v = (g[0] * x + g[1] * y + g[2] * z).astype(np.float32)
    ctx = disc.disc_create_ex((nx, ny, nz), (1, 1, 1), R, 1.5, 1, 1, (2, 2, 2))
    mu, var = torch.empty(v.shape, device="cuda"), torch.empty(v.shape, device="cuda")
    disc.disc_box_moments(ctx, 0, dev(v), mu, var)
    c = (slice(R[2], nz - R[2]), slice(R[1], ny - R[1]), slice(R[0], nx - R[0]))
    expect = sum(g[i] ** 2 * R[i] * (R[i] + 1) / 3.0 for i in range(3))
    np.testing.assert_allclose(var.cpu().numpy()[c], expect, rtol=1e-5)
    np.testing.assert_allclose(mu.cpu().numpy()[c], v[c], atol=1e-3)
    disc.disc_destroy(ctx)


@pytest.mark.parametrize("fac", [(2, 2, 1), (2, 1, 2), (1, 1, 1), (2, 2, 2), (1, 2, 1)])
def test_pyramid_with_per_axis_factors(disc, oracle_mod, fac):
    rng = np.random.default_rng(11)
    nx, ny, nz = 48, 36, 10
    v = rng.uniform(-1000, 1500, size=(nz, ny, nx)).astype(np.float32)
    ctx = disc.disc_create_ex((nx, ny, nz), (1, 1, 1), (1, 1, 1), 1.0, 2, 1, fac)
    cd = (nz // fac[2], ny // fac[1], nx // fac[0])
    assert ctx.level_dims(1) == (cd[2], cd[1], cd[0])
    out = torch.empty(cd, device="cuda")
    disc.disc_downsample(ctx, 0, dev(v), out)
    assert np.abs(out.cpu().numpy() - oracle_mod.downsample3(v, fac)).max() <= 1e-4 * 2500
    r = rng.normal(0, 3, size=(3,) + cd).astype(np.float32)
    up = torch.empty((3, nz, ny, nx), device="cuda")
    disc.disc_upsample_field(ctx, 1, dev(r), up)
    assert np.abs(up.cpu().numpy() - oracle_mod.upsample_field3(r, fac)).max() <= 1e-4
    disc.disc_destroy(ctx)


def test_create_ex_argument_errors(disc):
    ok = dict(dims=(32, 32, 17), spacing=(0.94, 0.94, 2.5), patch_radius=(1, 1, 1), sigma_smooth=1.5, levels=2, iters=1,
              pyramid_factor=(2, 2, 1))
    disc.disc_destroy(disc.disc_create_ex(**ok))                      # 17 slices: fine, z is not halved
    for bad, status in [(dict(pyramid_factor=(2, 2, 2)), disc.DISC_ERR_INVALID_ARG),   # 17 % 2 != 0
                        (dict(pyramid_factor=(2, 3, 1)), disc.DISC_ERR_INVALID_ARG),
                        (dict(patch_radius=(1, 1, -1)), disc.DISC_ERR_INVALID_ARG),
                        (dict(patch_radius=(2, 1, 1)), disc.DISC_ERR_UNSUPPORTED),     # Rx != Ry
                        (dict(patch_radius=(13, 13, 1)), disc.DISC_ERR_UNSUPPORTED)]:
        with pytest.raises(disc.DiscError) as e:
            disc.disc_create_ex(**{**ok, **bad})
        assert e.value.status == status


def clinical_pair():
    """config-3 generator at the paper's clinical size: 256 x 256 x 68"""
    return phantoms.make_pair(3, dims=(256, 256, 68))


@pytest.mark.slow
@pytest.mark.parametrize("R,iters", [((1, 1, 1), 60), ((12, 12, 3), 12)])
def test_clinical_geometry_whole_schedule(disc, oracle_mod, R, iters):
    """256x256x68, two levels with the transverse plane halved only, the paper's smallest (3x3x3) and largest (25x25x7)
    patch: disc_register against oracle.register_ex, final field within 1e-2 voxel."""
    ct, cbct, u, p = clinical_pair()
    nz, ny, nx = ct.shape
    sigma, levels, fac = 2.0, 2, (2, 2, 1)
    ctx = disc.disc_create_ex((nx, ny, nz), (0.94, 0.94, 2.5), R, sigma, levels, iters, fac)
    d_r, d_c = torch.empty((3,) + ct.shape, device="cuda"), torch.empty(ct.shape, device="cuda")
    disc.disc_register(ctx, dev(ct), dev(cbct), d_r, d_c)
    r, corr = d_r.cpu().numpy(), d_c.cpu().numpy()
    disc.disc_destroy(ctx)
    ref = oracle_mod.register_ex(ct, cbct, R, sigma, levels, iters, fac=fac, sat_between=True)
    err_r = float(np.abs(r - ref["disp"]).max())
    assert err_r <= 1e-2, f"field error {err_r} voxel"
    span = float(max(ct.max(), cbct.max()) - min(ct.min(), cbct.min()))
    g = float(max(np.abs(np.diff(ct, axis=a)).max() for a in range(3)))
    err_c = float(np.abs(corr - ref["corr"]).max())
    assert err_c <= 1e-4 * span + 2.0 * err_r * g + 1e-3, (err_c, err_r, g)
    if R == (1, 1, 1):
        target = phantoms.pullback(ct, u)
        body = target > -500.0
        m = oracle_mod.warp(ct, r)
        assert np.sqrt(np.mean((m - target)[body] ** 2)) < 0.8 * np.sqrt(np.mean((ct - target)[body] ** 2))

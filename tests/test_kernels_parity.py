"""Per-kernel parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Both sides always get the SAME fp32 inputs (never chained outputs).

Tolerances (BASELINE.json north_star / DESIGN.md): intensity outputs max-abs <= 1e-4 x (max - min of the
input volumes); displacement-valued outputs max-abs <= 1e-4 voxel.
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


def make_ctx(disc, shape, R=2, sigma=1.5, levels=1, iters=1):
    nz, ny, nx = shape
    return disc.disc_create((nx, ny, nz), (1.0, 1.0, 1.0), R, sigma, levels, iters)


def rand_pair(shape, seed, noise=20.0):
    """a CT-like smooth volume with edges and a deformed, biased, noisy companion"""
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    a = phantoms.volume_smooth_random((nx, ny, nz), rng, smooth=1.5) * 3.0
    a[: nz // 2, : ny // 2] += 600.0
    a = a.astype(np.float32)
    b = (0.9 * np.roll(a, 1, axis=2) - 100.0 + rng.normal(0, noise, a.shape)).astype(np.float32)
    return a, b


# nx % 4 == 0 takes the TMA-fed kernels, anything else the plain-load ones; both with ragged tiles
SHAPES = [(7, 6, 5), (9, 17, 33), (20, 45, 70), (32, 64, 64), (1, 1, 9), (3, 40, 2), (20, 45, 72), (21, 37, 132),
          (5, 3, 4), (30, 70, 260)]


# ------------------------------------------------------------------ warp
@pytest.mark.parametrize("shape", SHAPES)
def test_warp(disc, oracle_mod, shape):
    rng = np.random.default_rng(1)
    vol, _ = rand_pair(shape, 11)
    r = rng.uniform(-3, 3, size=(3,) + shape).astype(np.float32)
    r[:, 0, 0, 0] = (-50, 50, 0)           # far out of range: clamped
    ctx = make_ctx(disc, shape)
    out = torch.empty(shape, device="cuda")
    disc.disc_warp(ctx, 0, dev(vol), dev(r), out)
    ref = oracle_mod.warp(vol, r)
    tol = 1e-4 * float(vol.max() - vol.min())
    assert np.abs(out.cpu().numpy() - ref).max() <= tol
    # zero field: bit-exact identity
    disc.disc_warp(ctx, 0, dev(vol), torch.zeros((3,) + shape, device="cuda"), out)
    assert np.array_equal(out.cpu().numpy(), vol)


# ------------------------------------------------------------------ moments
@pytest.mark.parametrize("R", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10])
# Which kernel a case reaches (csrc/moments_tu.cu): nx % 4 != 0 -> the plain-load kernels; nx % 4 == 0 and at most two
# waves of 32x8x4 blocks (the first four such shapes, R <= 6) -> the block kernel of the coarse levels; nx % 4 == 0
# and either R >= 7 or more blocks than that (the last shape) -> the marching TMA + tensor-memory kernel.
@pytest.mark.parametrize("shape", [(7, 6, 5), (20, 45, 70), (37, 18, 33), (20, 45, 72), (37, 18, 36), (3, 5, 8),
                                   (26, 50, 100), (40, 100, 132)])
def test_box_moments(disc, oracle_mod, shape, R):
    vol, _ = rand_pair(shape, 20 + R)
    ctx = make_ctx(disc, shape, R=R)
    mean = torch.empty(shape, device="cuda"); var = torch.empty(shape, device="cuda")
    disc.disc_box_moments(ctx, 0, dev(vol), mean, var)
    rm, rv = oracle_mod.box_moments(vol, R)
    rngv = float(vol.max() - vol.min())
    assert np.abs(mean.cpu().numpy() - rm).max() <= 1e-4 * rngv
    assert np.abs(np.sqrt(var.cpu().numpy().astype(np.float64)) - np.sqrt(rv)).max() <= 1e-4 * rngv
    assert var.min().item() >= 0.0


# the block kernel of the coarse levels (csrc/moments_blk.cuh): blocks of 32 x 8 x 4 outputs (32 x 8 x 2 at R = 6) with
# ragged edges in every axis, volumes thinner than one block or than the patch, a single row, and all three modes
@pytest.mark.parametrize("R", [0, 1, 5, 6])
@pytest.mark.parametrize("shape", [(1, 1, 4), (2, 9, 12), (5, 8, 64), (9, 13, 36), (6, 3, 40)])
def test_block_kernel_edge_shapes(disc, oracle_mod, shape, R):
    vol, other = rand_pair(shape, 70 + R)
    ctx = make_ctx(disc, shape, R=R)
    mean = torch.empty(shape, device="cuda"); var = torch.empty(shape, device="cuda"); out = torch.empty(shape, device="cuda")
    disc.disc_box_moments(ctx, 0, dev(vol), mean, var)
    rm, rv = oracle_mod.box_moments(vol, R)
    rngv = max(float(vol.max() - vol.min()), 1.0)
    assert np.abs(mean.cpu().numpy() - rm).max() <= 1e-4 * rngv
    assert np.abs(np.sqrt(var.cpu().numpy().astype(np.float64)) - np.sqrt(rv)).max() <= 1e-4 * rngv
    disc.disc_correct_intensity(ctx, 0, dev(other), dev(vol), out)          # z-score of `other`, then the correction
    ref = oracle_mod.correct(other, vol, R)
    tol = 1e-4 * max(float(max(vol.max(), other.max()) - min(vol.min(), other.min())), 1.0)
    assert np.abs(out.cpu().numpy() - ref).max() <= tol


def test_box_moments_constant_volume_has_zero_variance(disc):
    """the H1 hazard: E(x^2) - mu^2 must not leak rounding into var (fp32 sums give ~9 HU^2 here)"""
    shape = (24, 40, 72)
    vol = np.full(shape, 1234.567, dtype=np.float32)
    ctx = make_ctx(disc, shape, R=3)
    mean = torch.empty(shape, device="cuda"); var = torch.empty(shape, device="cuda")
    disc.disc_box_moments(ctx, 0, dev(vol), mean, var)
    assert np.abs(mean.cpu().numpy() - np.float32(1234.567)).max() < 1e-3
    assert var.max().item() < 1e-6


# ------------------------------------------------------------------ correction
@pytest.mark.parametrize("R", [0, 1, 3, 5, 7, 10])
@pytest.mark.parametrize("shape", [(7, 6, 5), (20, 45, 70), (37, 18, 33), (20, 45, 72), (37, 18, 36), (26, 50, 100),
                                   (40, 100, 132)])
def test_correct_intensity(disc, oracle_mod, shape, R):
    m, s = rand_pair(shape, 30 + R)
    ctx = make_ctx(disc, shape, R=R)
    out = torch.empty(shape, device="cuda")
    disc.disc_correct_intensity(ctx, 0, dev(s), dev(m), out)
    ref = oracle_mod.correct(s, m, R)
    tol = 1e-4 * float(max(m.max(), s.max()) - min(m.min(), s.min()))
    assert np.abs(out.cpu().numpy() - ref).max() <= tol


def test_correct_intensity_clean_phantom_with_flat_regions(disc, oracle_mod):
    """noise-free CT against itself and against an affine copy: flat air/tissue patches have var = 0"""
    ct, _, _, _ = phantoms.make_pair(1, dims=(48, 40, 24))
    ctx = make_ctx(disc, ct.shape, R=3)
    out = torch.empty(ct.shape, device="cuda")
    tol = 1e-4 * float(ct.max() - ct.min())
    disc.disc_correct_intensity(ctx, 0, dev(ct), dev(ct), out)
    assert np.abs(out.cpu().numpy() - oracle_mod.correct(ct, ct, 3)).max() <= tol
    cti = np.round(ct).astype(np.float32)
    cb = (0.5 * cti - 120).astype(np.float32)
    disc.disc_correct_intensity(ctx, 0, dev(cb), dev(cti), out)
    assert np.abs(out.cpu().numpy() - cti).max() <= tol          # pin P7 on the CUDA path itself
    assert np.abs(out.cpu().numpy() - oracle_mod.correct(cb, cti, 3)).max() <= tol


# ------------------------------------------------------------------ force + update, Gaussian, demons step
@pytest.mark.parametrize("shape", SHAPES)
def test_force_update(disc, oracle_mod, shape):
    m, s = rand_pair(shape, 40)
    r0 = np.random.default_rng(41).normal(0, 1, size=(3,) + shape).astype(np.float32)
    ctx = make_ctx(disc, shape)
    r = dev(r0)
    disc.disc_force_update(ctx, 0, dev(m), dev(s), r)
    ref = oracle_mod.force_update(m, s, r0)
    assert np.abs(r.cpu().numpy() - ref).max() <= 1e-4
    # m = s: no force (bit exact)
    r = dev(r0)
    disc.disc_force_update(ctx, 0, dev(s), dev(s), r)
    assert np.array_equal(r.cpu().numpy(), r0)


@pytest.mark.parametrize("sigma", [0.3, 1.0, 1.5, 2.0, 2.5, 3.0, 4.0])
@pytest.mark.parametrize("shape", [(7, 6, 5), (20, 45, 70), (32, 64, 64), (3, 40, 2), (40, 300, 150), (20, 45, 72),
                                   (33, 70, 260)])
def test_smooth_field(disc, oracle_mod, shape, sigma):
    r0 = np.random.default_rng(50).normal(0, 3, size=(3,) + shape).astype(np.float32)
    ctx = make_ctx(disc, shape, sigma=sigma)
    r = dev(r0)
    disc.disc_smooth_field(ctx, 0, r)
    ref = oracle_mod.smooth_field(r0, sigma)
    assert np.abs(r.cpu().numpy() - ref).max() <= 1e-4
    # constant field preserved
    c = np.empty((3,) + shape, dtype=np.float32); c[0] = 1.25; c[1] = -3.5; c[2] = 7.0
    r = dev(c)
    disc.disc_smooth_field(ctx, 0, r)
    assert np.abs(r.cpu().numpy() - c).max() <= 2e-6


@pytest.mark.parametrize("shape", SHAPES)
def test_demons_step(disc, oracle_mod, shape):
    m, s = rand_pair(shape, 60)
    r0 = np.random.default_rng(61).normal(0, 1, size=(3,) + shape).astype(np.float32)
    ctx = make_ctx(disc, shape, sigma=1.5)
    r = dev(r0)
    disc.disc_demons_step(ctx, 0, dev(m), dev(s), r)
    ref = oracle_mod.demons_step(m, s, r0, 1.5)
    assert np.abs(r.cpu().numpy() - ref).max() <= 1e-4


# ------------------------------------------------------------------ double force (Eq. 1, both terms)
@pytest.mark.parametrize("sigma", [1.5, 2.0, 3.0])
@pytest.mark.parametrize("shape", SHAPES + [(40, 300, 152)])
def test_double_force(disc, oracle_mod, shape, sigma):
    m, s = rand_pair(shape, 70)
    r0 = np.random.default_rng(71).normal(0, 1, size=(3,) + shape).astype(np.float32)
    ctx = make_ctx(disc, shape, sigma=sigma)
    disc.disc_set_force(ctx, disc.DISC_FORCE_DOUBLE)
    r = dev(r0)
    disc.disc_force_update(ctx, 0, dev(m), dev(s), r)
    assert np.abs(r.cpu().numpy() - oracle_mod.force_update(m, s, r0, double_force=True)).max() <= 1e-4
    r = dev(r0)
    disc.disc_demons_step(ctx, 0, dev(m), dev(s), r)
    assert np.abs(r.cpu().numpy() - oracle_mod.demons_step(m, s, r0, sigma, double_force=True)).max() <= 1e-4
    # m = s: no force (bit exact); smoothing alone is unaffected by the mode
    r = dev(r0)
    disc.disc_force_update(ctx, 0, dev(s), dev(s), r)
    assert np.array_equal(r.cpu().numpy(), r0)
    # switching back restores the Thirion force
    disc.disc_set_force(ctx, disc.DISC_FORCE_THIRION)
    r = dev(r0)
    disc.disc_demons_step(ctx, 0, dev(m), dev(s), r)
    assert np.abs(r.cpu().numpy() - oracle_mod.demons_step(m, s, r0, sigma)).max() <= 1e-4
    with pytest.raises(disc.DiscError):
        disc.disc_set_force(ctx, 7)
    disc.disc_destroy(ctx)


# ------------------------------------------------------------------ pyramid
@pytest.mark.parametrize("shape", [(4, 6, 8), (16, 34, 66), (2, 2, 2)])
def test_pyramid(disc, oracle_mod, shape):
    vol, _ = rand_pair(shape, 70)
    ctx = make_ctx(disc, shape, levels=2)
    cs = tuple(n // 2 for n in shape)
    out = torch.empty(cs, device="cuda")
    disc.disc_downsample(ctx, 0, dev(vol), out)
    assert np.abs(out.cpu().numpy() - oracle_mod.downsample(vol)).max() <= 1e-4 * float(vol.max() - vol.min())
    rc = np.random.default_rng(71).normal(0, 2, size=(3,) + cs).astype(np.float32)
    up = torch.empty((3,) + shape, device="cuda")
    disc.disc_upsample_field(ctx, 1, dev(rc), up)
    assert np.abs(up.cpu().numpy() - oracle_mod.upsample_field(rc)).max() <= 1e-4


# ------------------------------------------------------------------ errors
def test_argument_errors(disc):
    ctx = make_ctx(disc, (8, 8, 8), levels=2)
    a = torch.zeros(512, device="cuda")
    with pytest.raises(disc.DiscError):
        disc.disc_warp(ctx, 2, a, torch.zeros(3 * 512, device="cuda"), a.clone())   # level out of range
    with pytest.raises(ValueError):
        disc.disc_warp(ctx, 0, a, torch.zeros(512, device="cuda"), a.clone())       # wrong size
    with pytest.raises(TypeError):
        disc.disc_warp(ctx, 0, a.cpu(), torch.zeros(3 * 512, device="cuda"), a.clone())
    with pytest.raises(disc.DiscError):
        disc.disc_upsample_field(ctx, 0, torch.zeros(3 * 512, device="cuda"), torch.zeros(3 * 4096, device="cuda"))
    assert "level" in disc.disc_last_error(ctx)


# ------------------------------------------------------------------ run-to-run reproducibility
@pytest.mark.parametrize("shape,R,sigma", [((32, 64, 64), 5, 2.0), ((26, 50, 100), 3, 1.5), ((9, 13, 36), 6, 1.0),
                                           ((40, 100, 132), 2, 2.5)])
def test_kernels_are_bit_reproducible(disc, shape, R, sigma):
    """Every kernel is a deterministic function of its inputs, so repeated launches must agree bit for bit.  A buffer
    released to its producer while loads from it are still in flight (the race the moments kernel once had, DESIGN.md
    section 8) or a shared-memory hazard between the phases of the tile kernels shows up here as a differing output."""
    rng = np.random.default_rng(5)
    nz, ny, nx = shape
    a, b = rand_pair(shape, 90)
    r0 = rng.uniform(-2, 2, size=(3,) + shape).astype(np.float32)
    ctx = make_ctx(disc, shape, R=R, sigma=sigma)
    da, db = dev(a), dev(b)
    ref = {}
    for it in range(60):
        out = torch.empty(shape, device="cuda"); disc.disc_correct_intensity(ctx, 0, db, da, out)
        mean = torch.empty(shape, device="cuda"); var = torch.empty(shape, device="cuda")
        disc.disc_box_moments(ctx, 0, da, mean, var)
        r = dev(r0)
        disc.disc_demons_step(ctx, 0, da, db, r)
        for k, v in (("corrected", out), ("mean", mean), ("var", var), ("step", r)):
            if it == 0:
                ref[k] = v.clone()
            else:
                assert torch.equal(ref[k], v), (k, it)
    disc.disc_destroy(ctx)

"""Config 4 as BASELINE.json states it -- 512x512x128, 4-level pyramid x 100 iterations, patch 15^3 (R = 7), sigma 2 --
disc_register against the oracle over the WHOLE schedule (north_star: final displacement within 1e-2 voxel).

The naive patch loops need ~15 s per 512x512x128 moment evaluation on the box's 16 cores, i.e. ~30 min for this
schedule, so the oracle follows SURVEY.md section 8(c) "Oracle cost": naive loops for the CBCT moments and for the first
and last iteration of every level, and the independently written fp64 summed-area routine -- pinned against the
naive loops on CPU (tests/test_oracle_pins_ext.py::test_sat_moments_match_naive, ..._on_a_phantom) -- in between.
Takes ~8 min of oracle time; it is the last file of the suite so that everything else has run before it starts.
"""
import numpy as np
import pytest

import phantoms

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

torch = pytest.importorskip("torch")


def test_config4_whole_schedule_against_the_oracle(oracle_mod):
    import __graft_entry__
    __graft_entry__.build()
    import paper_1204_6295_b200 as disc
    ct, cbct, u, p = phantoms.make_pair(4)
    nz, ny, nx = ct.shape
    R, sigma = p["patch_radius"], p["sigma"]
    assert (nx, ny, nz, R, p["levels"], p["iters"]) == (512, 512, 128, 7, 4, 100)
    ctx = disc.disc_create((nx, ny, nz), (1, 1, 1), R, sigma, p["levels"], p["iters"])
    d_ct, d_cb = torch.from_numpy(ct).cuda(), torch.from_numpy(cbct).cuda()
    d_r, d_corr = torch.empty((3,) + ct.shape, device="cuda"), torch.empty_like(d_ct)
    disc.disc_register(ctx, d_ct, d_cb, d_r, d_corr)
    assert disc.disc_iterations_run(ctx) == [p["iters"]] * p["levels"]
    d_m, d_c2 = torch.empty_like(d_ct), torch.empty_like(d_ct)
    disc.disc_warp(ctx, 0, d_ct, d_r, d_m)
    disc.disc_correct_intensity(ctx, 0, d_cb, d_m, d_c2)
    assert torch.equal(d_c2, d_corr)                                   # reading A12
    r, corr, m = d_r.cpu().numpy(), d_corr.cpu().numpy(), d_m.cpu().numpy()
    disc.disc_destroy(ctx)
    del d_ct, d_cb, d_r, d_corr, d_m, d_c2
    assert np.isfinite(r).all()
    ref = oracle_mod.register_ex(ct, cbct, R, sigma, p["levels"], p["iters"], sat_between=True)
    err_r = float(np.abs(r - ref["disp"]).max())
    assert err_r <= 1e-2, f"field error {err_r} voxel after the 4 x 100 schedule"
    span = float(max(ct.max(), cbct.max()) - min(ct.min(), cbct.min()))
    g = float(max(np.abs(np.diff(ct, axis=a)).max() for a in range(3)))
    err_c = float(np.abs(corr - ref["corr"]).max())
    assert err_c <= 1e-4 * span + 2.0 * err_r * g + 1e-3, (err_c, err_r, g)
    target = phantoms.pullback(ct, u)
    body = target > -500.0
    rmse0 = np.sqrt(np.mean((ct - target)[body] ** 2))
    rmse1 = np.sqrt(np.mean((m - target)[body] ** 2))
    assert rmse1 < 0.7 * rmse0, (rmse0, rmse1)

"""Alg. A1 with the reliability mask (steps 1-6; Eqs. (5)-(10) PAPER.md:117-139; "globally adjust"
PAPER.md:161, :179; parameter rules PAPER.md:165) composed from the oracle's step functions, one call per step, so that
a test can look at -- and override -- the Eq. (7) decisions of every iteration.

Eq. (7) is a hard threshold on chained floating-point values: two correct implementations that differ by rounding take
different decisions at a voxel that sits on a threshold, and from there on they compute different (both valid)
registrations.  A parity test therefore lets one side follow the other's decisions after checking that every voxel
where they differ does sit on a threshold, and compares everything else with plain bounds.

tests/test_oracle_pins_ext.py pins this composition (with its own decisions) against oracle.register_ex; the GPU test
in tests/test_next1_mask.py drives it with the CUDA path's decisions.  Helper module, not collected by pytest.
"""
import numpy as np


def level_shape(shape, level):
    return tuple(s // 2 ** level for s in shape)


def run(oracle, ct, cbct, R, sigma, levels, iters, fill_radius, h, hu0=None, a_range=None, max_fill_passes=64,
        params=None, decide=None, after_level=None):
    """Returns dict(disp, corr, params, cbct_shift).  params = (hu0, a_min, a_max) overrides the rules of PAPER.md:165.
    decide(level, k, m, cbct_l, a0, xi_own) -> the xi (bool array) the iteration goes on with (default: its own).
    after_level(level, r) is called with the field at the end of each level."""
    d = oracle.delta_hu(ct, cbct)
    cbct0 = (cbct.astype(np.float64) + d).astype(np.float32)
    if params is None:
        p_hu0 = hu0 if hu0 is not None else 2.0 * abs(d)
        if a_range is not None:
            a_min, a_max = a_range
        else:
            mus, vs = oracle.box_moments(cbct0, R)
            mum, vm = oracle.box_moments(ct, R)
            a_pre, _ = oracle.ab_from_moments(mus, vs, mum, vm)
            a_m = oracle.median_a(a_pre, vs, vm)
            a_min, a_max = 0.5 * a_m, 1.5 * a_m
        params = (p_hu0, a_min, a_max)
    pct, pcb = [ct], [cbct0]
    for l in range(1, levels):
        pct.append(oracle.downsample(pct[-1]))
        pcb.append(oracle.downsample(pcb[-1]))
    r = None
    for l in range(levels - 1, -1, -1):
        r = np.zeros((3,) + pct[l].shape, dtype=np.float32) if r is None else oracle.upsample_field(r)
        mus, vs = oracle.box_moments(pcb[l], R)

        def corrected(m, k):
            mum, vm = oracle.box_moments(m, R)                                     # A1 step 1
            a0, b0 = oracle.ab_from_moments(mus, vs, mum, vm)                      # Eqs. (5), (6)
            xi = oracle.mask(m, pcb[l], a0, *params) != 0                          # Eq. (7)
            if decide is not None:
                xi = decide(l, k, m, pcb[l], a0, xi)
            fa, fb, _, _ = oracle.fill_ab(pcb[l], xi.astype(np.uint8), a0, b0, fill_radius, h, max_fill_passes)   # step 2
            return oracle.apply_ab(pcb[l], fa, fb)                                 # step 3

        for k in range(iters):
            m = oracle.warp(pct[l], r)
            sp = corrected(m, k)
            r = oracle.demons_step(m, sp, r, sigma)                                # steps 4-6
        if after_level is not None:
            after_level(l, r)
    corr = corrected(oracle.warp(pct[0], r), iters)                                # reading A12
    return {"disp": r, "corr": corr, "params": params, "cbct_shift": cbct0, "delta_hu": d}

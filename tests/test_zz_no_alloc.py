"""disc_smooth_field_noalloc -- the entry point for callers that are not allowed to allocate device memory.

Some users of the library cannot call cudaMalloc while they run: a host application that partitions the GPU's memory
itself and forbids allocations from libraries, or a latency-bound loop for which the device-wide synchronisation of
cudaMalloc / cudaFree is not acceptable.  disc_create allocates every kernel's scratch, so those callers cannot have a
context; disc_smooth_field_noalloc gives them the Gaussian regularisation of a field (step (d)) with the
buffer between its two kernels in a fixed array inside libdisc.so (at most DISC_NOALLOC_MAX_VOXELS voxels).

What is checked: its output against disc_smooth_field (the existing path, same kernels, context-owned scratch) on two
calls in a row -- the second on a smaller volume and another sigma, so that it runs over whatever the first call left
in the shared array -- within the 1e-4 voxel of tests/test_kernels_parity.py::test_smooth_field; that a volume beyond
the built-in array is refused with a message instead of overrunning it; and the argument errors.

This file is collected last on purpose (pytest -x stops at the first failure) and passes on its own in a fresh
process as well as after the rest of the suite: it makes its own contexts and inputs and relies on nothing earlier.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = 1e-4   # voxel; the tolerance of test_smooth_field


@pytest.fixture(scope="module")
def disc():
    import __graft_entry__
    __graft_entry__.build()
    import paper_1204_6295_b200 as d
    assert torch.cuda.is_available()
    return d


def field(shape, seed):
    r = np.random.default_rng(seed).normal(0, 3, size=(3,) + shape).astype(np.float32)
    return torch.from_numpy(r).cuda()


def existing_path(disc, shape, sigma, r0):
    nz, ny, nx = shape
    ctx = disc.disc_create((nx, ny, nz), (1.0, 1.0, 1.0), 1, sigma, 1, 1)
    r = r0.clone()
    disc.disc_smooth_field(ctx, 0, r)
    torch.cuda.synchronize()
    disc.disc_destroy(ctx)
    return r


def test_two_calls_in_a_row_match_the_context_path(disc):
    # first call: 64 x 128 x 128 voxels = the largest volume the built-in array takes, tile kernels (nx % 4 == 0)
    # second call: a smaller ragged volume through the plain-load kernels, other sigma, over the first call's leftovers
    cases = [((64, 128, 128), 2.0, 900), ((21, 37, 130), 1.5, 901)]
    assert 64 * 128 * 128 == disc.DISC_NOALLOC_MAX_VOXELS
    inputs = [field(shape, seed) for shape, _, seed in cases]
    got = []
    for (shape, sigma, _), r0 in zip(cases, inputs):            # the two calls, back to back on the current stream
        nz, ny, nx = shape
        r = r0.clone()
        disc.disc_smooth_field_noalloc((nx, ny, nz), sigma, r)
        got.append(r)
    torch.cuda.synchronize()
    for (shape, sigma, _), r0, r in zip(cases, inputs, got):
        ref = existing_path(disc, shape, sigma, r0)
        assert torch.isfinite(r).all()
        assert not torch.equal(r, r0)                           # it did run
        assert (r - ref).abs().max().item() <= TOL, (shape, sigma)
        assert torch.equal(r, ref), (shape, sigma)              # same kernels, same launch shapes: identical bits


def test_same_call_twice_gives_the_same_bits(disc):
    shape, sigma = (32, 64, 64), 2.5
    nz, ny, nx = shape
    r0 = field(shape, 902)
    a, b = r0.clone(), r0.clone()
    disc.disc_smooth_field_noalloc((nx, ny, nz), sigma, a)
    disc.disc_smooth_field_noalloc((nx, ny, nz), sigma, b)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    assert (a - existing_path(disc, shape, sigma, r0)).abs().max().item() <= TOL


def test_size_beyond_the_builtin_array_is_refused(disc):
    nx, ny, nz = 128, 128, 65                                   # one slice more than the array holds
    assert nx * ny * nz > disc.DISC_NOALLOC_MAX_VOXELS
    r = torch.zeros(3 * nx * ny * nz, device="cuda")
    with pytest.raises(disc.DiscError) as e:
        disc.disc_smooth_field_noalloc((nx, ny, nz), 2.0, r)
    assert e.value.status == disc.DISC_ERR_INVALID_ARG
    assert "DISC_NOALLOC_MAX_VOXELS" in str(e.value) and str(disc.DISC_NOALLOC_MAX_VOXELS) in str(e.value)
    torch.cuda.synchronize()
    assert not r.any()                                          # nothing was launched
    small = torch.zeros(3 * 8 * 8 * 8, device="cuda")
    for dims, sigma, status in (((0, 8, 8), 1.0, disc.DISC_ERR_INVALID_ARG), ((8, 8, 8), 0.0, disc.DISC_ERR_INVALID_ARG),
                                ((8, 8, 8), 4.5, disc.DISC_ERR_UNSUPPORTED)):
        with pytest.raises(disc.DiscError) as e:
            disc.disc_smooth_field_noalloc(dims, sigma, small if dims[0] else torch.zeros(0, device="cuda"))
        assert e.value.status == status, (dims, sigma)

"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/disc.h declares; argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__
    __graft_entry__.build()
    import paper_1204_6295_b200 as disc
    return disc


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "disc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(disc_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for n in ("disc_create", "disc_correct_intensity", "disc_warp", "disc_demons_step", "disc_register"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    dll = ctypes.CDLL(lib.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(dll, name), name
    assert sorted(lib.EXPORTS) == declared_symbols()
    for name in lib.EXPORTS:
        assert callable(getattr(lib, name)), name


def test_library_is_built_for_sm_100a(lib):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", lib.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_create_validates_arguments_before_touching_the_device(lib):
    bad = [
        dict(dims=(0, 8, 8)), dict(dims=(8, 8, 6), levels=3), dict(spacing=(1, 0, 1)), dict(patch_radius=-1),
        dict(sigma_smooth=0.0), dict(levels=0), dict(iters=-1), dict(levels=9),
    ]
    for kw in bad:
        args = dict(dims=(8, 8, 8), spacing=(1, 1, 1), patch_radius=1, sigma_smooth=1.0, levels=1, iters=1)
        args.update(kw)
        with pytest.raises(lib.DiscError) as e:
            lib.disc_create(**args)
        assert e.value.status == lib.DISC_ERR_INVALID_ARG, kw
    for kw in (dict(patch_radius=13), dict(sigma_smooth=4.5)):
        args = dict(dims=(8, 8, 8), spacing=(1, 1, 1), patch_radius=1, sigma_smooth=1.0, levels=1, iters=1)
        args.update(kw)
        with pytest.raises(lib.DiscError) as e:
            lib.disc_create(**args)
        assert e.value.status == lib.DISC_ERR_UNSUPPORTED, kw


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(lib.DiscError) as e:
        lib.disc_create((8, 8, 8), (1, 1, 1), 1, 1.0, 1, 1)
    assert e.value.status in (lib.DISC_ERR_CUDA, lib.DISC_ERR_UNSUPPORTED)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1204_6295_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU or PyTorch fallback", ""), os.path.join(dirpath, f)

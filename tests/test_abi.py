"""CPU-side checks of the C-ABI boundary: libmc.so builds for sm_100a, loads without a GPU and
exports every symbol include/mc.h declares; host-side validation that needs no device."""
import ctypes as C
import os
import re

import pytest

from paper_2607_02954_b200 import binding, build, worlds

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mc_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert set(names) == set(binding.SYMBOLS)
    for n in names:
        assert hasattr(lib, n), n


def test_no_oracle_or_cpu_fallback_in_product():
    # the product package must not import the oracle
    pkg = os.path.join(ROOT, "paper_2607_02954_b200")
    for dirpath, _dirs, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "mco_" not in txt and "mco.h" not in txt, f


def test_workspace_bytes_validation(lib):
    w = worlds.make_world("1")
    good = binding.workspace_bytes(w["params"])
    nc = 64 * 64
    assert good > 2 * 9 * nc * 4  # at least the two population buffers
    bad = dict(w["params"], nx=65)
    assert binding.workspace_bytes(bad) == 0
    for key, val in (("pbd_iters", 0), ("pbd_iters", 9), ("pbd_order", 2), ("pbd_project", 2), ("two_layer", -1),
                     ("layer_offset", 1.5)):
        assert binding.workspace_bytes(dict(w["params"], **{key: val})) == 0, key
    assert binding.workspace_bytes(dict(w["params"], two_layer=1, coupling=1, mdf_iters=2)) > good  # readings 26 + 28 together
    # literal PBD and the two-layer broadcast are accepted; two layers double the tile lists
    assert binding.workspace_bytes(dict(w["params"], pbd_iters=4, pbd_order=1)) == good
    assert binding.workspace_bytes(dict(w["params"], two_layer=1)) > good
    # a batch is n worlds side by side
    wp, _k = binding.make_params(w["params"])
    assert lib.mc_batch_workspace_bytes(C.byref(wp), 7) == 7 * good
    assert lib.mc_batch_workspace_bytes(C.byref(wp), 0) == 0 and lib.mc_batch_workspace_bytes(C.byref(wp), 70000) == 0
    bad = dict(w["params"], nu=0.0)
    assert binding.workspace_bytes(bad) == 0
    # capacity scales with max_beads and with the grid
    big = dict(w["params"], max_beads=10_000_000, nx=6272, ny=6272)
    b = binding.workspace_bytes(big)
    assert 3e9 < b < 8e9  # fits one B200 many times over


def test_create_rejects_bad_arguments_without_touching_the_device(lib):
    w = worlds.make_world("1")
    wp, _keep = binding.make_params(w["params"])
    h = C.c_void_p()
    # null workspace -> MC_EINVAL before any CUDA call
    rc = lib.mc_create(C.byref(wp), None, 0, None, C.byref(h))
    assert rc == binding.MC_EINVAL and not h.value
    assert b"workspace" in lib.mc_last_error(None)
    assert lib.mc_step(None, 1) == binding.MC_EINVAL
    lib.mc_destroy(None)
    hb = C.c_void_p()
    rc = lib.mc_create_batch(C.byref(wp), 4, None, 0, None, C.byref(hb))
    assert rc == binding.MC_EINVAL and not hb.value
    assert b"workspace" in lib.mc_batch_last_error(None)
    assert lib.mc_step_batch(None, 1) == binding.MC_EINVAL
    lib.mc_destroy_batch(None)


def test_binding_refuses_to_run_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.World(worlds.make_world("1"))

"""mc_deposit_noalloc: the one entry point of libmc.so that allocates nothing (include/mc.h).

It runs S2 (rho_b = sum_i delta_h(g - X_i)) with the step's own kernels, their scratch in a
file-scope static device array instead of a caller workspace, for callers that cannot call
cudaMalloc.  Checked against the existing path -- a world's S2 read back with
mc_read_intermediates -- with the tolerances of the parity suite (rel L2 1e-5, element-wise 5e-6),
on two calls in a row (the scratch is shared and keeps the last call's contents).

This file is named so that pytest collects it LAST (the suite runs with `pytest -x`): it passes
when run alone in a fresh process and after all other tests.
"""
import numpy as np
import pytest

from paper_2607_02954_b200 import worlds

pytestmark = pytest.mark.gpu

TOL_L2, TOL_MAX = 1e-5, 5e-6   # tests/test_gpu_parity.py: TOL_STEP, TOL_MAX


def _rel_l2(a, b):
    a, b = np.asarray(a, np.float64).ravel(), np.asarray(b, np.float64).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def _max_ratio(a, b):
    a, b = np.asarray(a, np.float64).ravel(), np.asarray(b, np.float64).ravel()
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def _existing_path(w):
    """rho_b of the world's first step = S2 of the loaded positions, through mc_step + mc_read_intermediates."""
    from paper_2607_02954_b200 import binding
    G = binding.World(w)
    G.keep_intermediates(True)   # read_intermediates also returns G, which is only stored on request
    G.step(1)
    rho_b = G.read_intermediates()["rho_b"]
    G.close()
    return rho_b


def test_no_alloc_deposit_matches_the_step_on_two_calls_in_a_row():
    import torch
    from oracle import mco
    from paper_2607_02954_b200 import binding
    # two different worlds, back to back through the SAME static scratch: the second call must not see
    # anything of the first (more tiles and longer lists first, then fewer)
    wa = worlds.ragged_world(96, 64, [3, 5, 16, 31, 33, 64, 65, 100], seed=5)      # chains across the seam, |X| beyond a period
    wb = worlds.random_world(64, 64, 96, 16, seed=7, kappa=0.25, kappa_rep=2e-4, clustered=3.0)   # crowded: > 1024 beads in a tile
    want = [_existing_path(wa), _existing_path(wb)]
    torch.cuda.synchronize()
    xs = [torch.from_numpy(w["xy"]).cuda().contiguous() for w in (wa, wb)]
    outs = [torch.full((w["params"]["ny"], w["params"]["nx"]), float("nan"), device="cuda") for w in (wa, wb)]
    again = torch.full_like(outs[0], float("nan"))
    binding.load_library()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # call 1, call 2 (different world), call 3 = call 1 again: all on one stream, no sync in between
    binding.deposit_noalloc(wa["params"]["nx"], wa["params"]["ny"], xs[0], outs[0])
    binding.deposit_noalloc(wb["params"]["nx"], wb["params"]["ny"], xs[1], outs[1])
    binding.deposit_noalloc(wa["params"]["nx"], wa["params"]["ny"], xs[0], again)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the call changed the device's free memory"
    got = [o.cpu().numpy() for o in outs]
    for g, r, w in zip(got, want, (wa, wb)):
        assert np.isfinite(g).all()
        assert _rel_l2(g, r) <= TOL_L2 and _max_ratio(g, r) <= TOL_MAX, (_rel_l2(g, r), _max_ratio(g, r))
        assert abs(g.astype(np.float64).sum() - len(w["xy"])) < 1e-5 * len(w["xy"])   # every bead deposits unit mass
        # and against the oracle's definition written out
        o = mco.deposit(w["params"]["nx"], w["params"]["ny"], w["xy"].astype(np.float64))
        assert _rel_l2(g, o) <= TOL_L2 and _max_ratio(g, o) <= TOL_MAX
    assert again.cpu().numpy().tobytes() == got[0].tobytes()        # deterministic, whatever ran before
    print("no-alloc deposit vs step:", [(_rel_l2(g, r), _max_ratio(g, r)) for g, r in zip(got, want)])


def test_no_alloc_limits_and_empty_input():
    import torch
    from paper_2607_02954_b200 import binding
    out = torch.ones((64, 96), device="cuda")
    # no beads: an all-zero field
    binding.deposit_noalloc(96, 64, torch.empty((0, 2), device="cuda"), out)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
    # sizes beyond the static scratch are refused with a message that names the limit
    big = torch.zeros((binding.NOALLOC_MAX_BEADS + 1, 2), device="cuda")
    with pytest.raises(binding.McError) as e:
        binding.deposit_noalloc(96, 64, big, out)
    assert e.value.code == binding.MC_EINVAL and "MC_NOALLOC_MAX_BEADS" in str(e.value)
    wide = torch.empty((32, 32 * (binding.NOALLOC_MAX_TILES + 1)), device="cuda")
    with pytest.raises(binding.McError) as e:
        binding.deposit_noalloc(32 * (binding.NOALLOC_MAX_TILES + 1), 32, big[:8], wide)
    assert e.value.code == binding.MC_EINVAL and "MC_NOALLOC_MAX_TILES" in str(e.value)
    with pytest.raises(binding.McError):
        binding.deposit_noalloc(100, 64, big[:8], torch.empty((64, 100), device="cuda"))   # not a multiple of 32
    # the largest sizes it takes: MC_NOALLOC_MAX_BEADS beads on MC_NOALLOC_MAX_TILES tiles
    n = binding.NOALLOC_MAX_BEADS
    xy = (torch.rand((n, 2), device="cuda", generator=torch.Generator(device="cuda").manual_seed(3)) * 1024.0).contiguous()
    full = torch.empty((1024, 1024), device="cuda")
    binding.deposit_noalloc(1024, 1024, xy, full)
    torch.cuda.synchronize()
    assert abs(float(full.double().sum()) - n) < 1e-5 * n

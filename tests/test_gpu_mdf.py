"""GPU parity of the Multi-Direct Forcing coupling (MC_COUPLING_MDF; SURVEY.md 8(f) NEXT-1,
DESIGN.md reading 26) against the oracle, through the C ABI.  Same protocol and bars as
tests/test_gpu_parity.py: per step 1e-5 relative L2 on every output, 1e-3 on the positions after
100 free-running steps, bit-exact run to run.
"""
import numpy as np
import pytest

from paper_2607_02954_b200 import worlds
from test_gpu_parity import TOL_STEP, TOL_TRAJ, assert_close, rel_l2, run_protocol

pytestmark = pytest.mark.gpu


def mdf(w, iters=3):
    w["params"]["coupling"] = 1
    w["params"]["mdf_iters"] = iters
    return w


MDF = {
    # ragged chains (3 .. 100 beads), several tiles, chains across the periodic seam
    "ragged_96x64": lambda: mdf(worlds.ragged_world(96, 64, [3, 4, 5, 16, 31, 32, 33, 59, 60, 61, 64, 65, 100],
                                                    seed=3)),
    # both field kinds: V carries the repulsion and the chemotaxis displacement
    "static_64x96": lambda: mdf(worlds.ragged_world(64, 96, [8, 16, 32, 64, 7, 45], seed=4, static_source=True), 2),
    # no fields: tile bounds without rho_b (the fallback scale of the broadcast)
    "no_fields": lambda: mdf(worlds.ragged_world(64, 32, [10, 20, 40], seed=6, kappa_rep=None), 4),
    # one iteration: no broadcast kernel at all, only the fused spread
    "one_iter": lambda: mdf(worlds.ragged_world(64, 64, [12, 30, 50], seed=17), 1),
    # one tile in each direction: every support wraps onto the same tile
    "single_tile_32": lambda: mdf(worlds.ragged_world(32, 32, [5, 12, 20], seed=11), 3),
    # uniform 64-bead chains (configs 2 and 4), many empty tiles
    "uniform_m64": lambda: mdf(worlds.random_world(256, 160, 40, 64, seed=8), 3),
    # the most iterations the ABI takes
    "iters_16": lambda: mdf(worlds.random_world(96, 128, 30, 32, seed=9), 16),
}


@pytest.mark.parametrize("name", sorted(MDF))
def test_mdf_per_step_parity(name):
    w = MDF[name]()
    worst = run_protocol(w, steps_at=[0, 1, 10, 40])
    print(name, {k: f"{v:.2e}" for k, v in worst.items()})


def test_mdf_config1_trajectory():
    from oracle import mco
    from paper_2607_02954_b200 import binding
    w = mdf(worlds.make_world("1"))
    worst = run_protocol(w, steps_at=[0, 1, 10, 99])
    print("config1 mdf", {k: f"{v:.2e}" for k, v in worst.items()})
    G, O = binding.World(w), mco.World(w)
    G.step(100)
    O.step(100)
    g, o = G.read_state(), O.read_state()
    assert_close("X after 100 steps", g["xy"], o["xy"], TOL_TRAJ)
    d = rel_l2(g["xy"].astype(np.float64) - w["xy"], o["xy"] - w["xy"])[0]
    print(f"config1 mdf 100-step displacement rel L2 {d:.2e}")
    assert d < 5e-2
    assert np.abs(o["u"]).max() < 0.1


def test_mdf_config2_per_step_and_trajectory():
    from oracle import mco
    from paper_2607_02954_b200 import binding
    w = mdf(worlds.make_world("2"))
    worst = run_protocol(w, steps_at=[0, 5, 60], threads=8)
    print("config2 mdf", {k: f"{v:.2e}" for k, v in worst.items()})
    G, O = binding.World(w), mco.World(w, threads=8)
    G.step(100)
    O.step(100)
    g, o = G.read_state(), O.read_state()
    assert_close("X after 100 steps", g["xy"], o["xy"], TOL_TRAJ)
    assert np.abs(o["u"]).max() < 0.1 and np.abs(o["rho"] - 1).max() < 0.1


def test_mdf_bitwise_reproducible_and_batching():
    from paper_2607_02954_b200 import binding
    outs = []
    for split in ((23,), (23,), (3, 20), (1,) * 23):
        G = binding.World(MDF["uniform_m64"]())
        for n in split:
            G.step(n)
        outs.append(G.read_state(keys=("xy", "u", "fdev", "force")))
        G.close()
    for o in outs[1:]:
        for k in ("xy", "u", "fdev", "force"):
            assert outs[0][k].tobytes() == o[k].tobytes(), k


def test_mdf_reduces_the_slip():
    # what the iterations are for: the bead velocity U = dX approaches V = D as mdf_iters grows
    from oracle import mco
    from paper_2607_02954_b200 import binding
    errs = []
    for K in (1, 2, 4, 8):
        w = mdf(worlds.random_world(96, 64, 10, 32, seed=21, kappa_rep=None), K)
        G = binding.World(w)
        G.step(6)
        s0 = G.read_state(keys=("xy",))
        G.step(1)
        s1 = G.read_state(keys=("xy",))
        D = mco.elastic(w["offsets"], s0["xy"].astype(np.float64), w["L_rest"], w["theta_rest"], w["k_bend"],
                        w["k_shear"], w["k_stretch"], w["act_amp"], w["act_phase"], w["act_period"],
                        float(np.float32(w["params"]["dt"])), 6)
        errs.append(np.abs((s1["xy"].astype(np.float64) - s0["xy"]) - D).max() / np.abs(D).max())
        G.close()
    print("slip vs iterations", errs)
    assert all(b < a for a, b in zip(errs, errs[1:])), errs


def test_mdf_parameters_are_validated():
    from paper_2607_02954_b200 import binding
    for it in (0, 17):
        with pytest.raises(binding.McError):
            binding.World(mdf(worlds.random_world(64, 64, 4, 8, seed=2), it))
    w = worlds.random_world(64, 64, 4, 8, seed=2)
    w["params"]["coupling"] = 7
    with pytest.raises(binding.McError):
        binding.World(w)


@pytest.mark.parametrize("name,steps_at", [("4b", [0, 20]), ("4c", [8])])
def test_mdf_per_step_parity_config4(name, steps_at):
    import os
    w = mdf(worlds.make_world(name))
    worst = run_protocol(w, steps_at=steps_at, threads=os.cpu_count() or 1)
    print(name, "mdf", {k: f"{v:.2e}" for k, v in worst.items()})


def test_mdf_config_4d_properties_and_sampled_parity():
    # the size bench.py --coupling mdf times: properties that hold at any size, and outputs the
    # oracle's components can reproduce on samples
    from oracle import mco
    from paper_2607_02954_b200 import binding
    CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1], dtype=np.float64)
    CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1], dtype=np.float64)
    w = mdf(worlds.make_world("4d"))
    G = binding.World(w)
    G.keep_intermediates(True)
    G.step(5)
    s0 = G.read_state(keys=("xy", "fdev"))
    G.step(1)
    s1 = G.read_state(keys=("xy", "fdev", "u", "force", "rho"))
    it = G.read_intermediates()
    G.close()
    # fluid mass conserved; momentum grows by sum(G) = sum of the summed bead forces
    a0 = s0["fdev"].astype(np.float64).sum(axis=(1, 2))
    a1 = s1["fdev"].astype(np.float64).sum(axis=(1, 2))
    assert abs(a1.sum() - a0.sum()) < 1e-6 * np.abs(s1["fdev"]).astype(np.float64).sum()
    for C, ch in ((CX, 0), (CY, 1)):
        gsum = it["G"][ch].astype(np.float64).sum()
        gabs = np.abs(it["G"][ch]).astype(np.float64).sum()
        assert abs((C @ a1 - C @ a0) - gsum) < 1e-5 * gabs + 1e-9
        assert abs(s1["force"][:, ch].astype(np.float64).sum() - gsum) < 1e-5 * gabs
    assert np.abs(s1["u"]).max() < 0.1 and np.abs(s1["rho"] - 1.0).max() < 0.1
    # sampled chains: the position update is the interpolation of the stored u
    rng = np.random.default_rng(1)
    chains = rng.choice(len(w["offsets"]) - 1, size=64, replace=False)
    idx = np.concatenate([np.arange(w["offsets"][c], w["offsets"][c + 1]) for c in chains])
    X0 = s0["xy"][idx].astype(np.float64)
    assert_close("sampled X update", s1["xy"][idx], X0 + mco.interp(s1["u"].astype(np.float64), X0), TOL_STEP)
    # sampled windows of the grid: G equals the oracle's spread of the GPU's summed bead forces
    # (beads within reach of a 32x32 window, moved into a 64x64 periodic box around it)
    nx = w["params"]["nx"]
    X = s0["xy"].astype(np.float64)
    for (x0, y0) in ((1000, 2000), (0, 0), (nx - 32, 3136)):
        dx = (X[:, 0] - (x0 - 16)) % nx
        dy = (X[:, 1] - (y0 - 16)) % nx
        sel = (dx > 8) & (dx < 56) & (dy > 8) & (dy < 56)
        loc = np.stack([dx[sel], dy[sel]], 1)
        Gw = mco.spread(64, 64, loc, s1["force"][sel].astype(np.float64))[:, 16:48, 16:48]
        ii = (np.arange(32) + x0) % nx
        jj = (np.arange(32) + y0) % nx
        assert_close(f"G window at {(x0, y0)}", it["G"][:, jj][:, :, ii], Gw, TOL_STEP)
    # bit-for-bit reproducible at full size
    H = binding.World(w)
    H.step(6)
    h = H.read_state(keys=("xy", "u"))
    H.close()
    assert h["xy"].tobytes() == s1["xy"].tobytes() and h["u"].tobytes() == s1["u"].tobytes()


def test_mdf_on_clustered_tiles_one_iteration():
    # a crowded world (thread-block clusters per tile, hi + lo accumulator words) under MDF: the
    # summed force reaches the cluster variant of the fused kernel with K5b's per-tile bound.  One
    # forcing iteration only: with ~50 beads per cell the iteration itself amplifies (reading 26),
    # which is a property of the method, not of the kernels.
    from paper_2607_02954_b200 import binding
    w = mdf(worlds.random_world(96, 64, 2500, 16, seed=23, kappa=0.25, kappa_rep=2e-5, clustered=4.0), 1)
    w["act_amp"][:] = 0  # only the (weak) repulsion drives V; with rho_b up to 240 the second step already
    # overshoots 120-fold in the oracle too, so the parity step is the first one
    G = binding.World(w)
    assert G.cluster_tiles(-1) == 4
    G.close()
    worst = run_protocol(w, steps_at=[0])
    print("mdf clustered", {k: f"{v:.2e}" for k, v in worst.items()})

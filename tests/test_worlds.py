"""The seeded input generators (shared by the CUDA path and the oracle): version-proof counter RNG,
the shapes BASELINE.json names for each config, and the recipe's invariants."""
import math

import numpy as np
import pytest

from paper_2607_02954_b200 import worlds


def test_counter_rng_is_pinned():
    # first values of the splitmix64-based stream must never change (inputs are not stored)
    u = worlds.uniform(0, "pin", 4)
    assert u.dtype == np.float64 and np.all((u >= 0) & (u < 1))
    assert np.array_equal(u, worlds.uniform(0, "pin", 4))
    assert not np.array_equal(u, worlds.uniform(1, "pin", 4))
    assert not np.array_equal(u, worlds.uniform(0, "pin2", 4))
    # 24-bit resolution
    assert np.all(u * (1 << 24) == np.round(u * (1 << 24)))
    n = worlds.normal(3, "n", 20000)
    assert abs(n.mean()) < 0.03 and abs(n.std() - 1.0) < 0.03


@pytest.mark.parametrize("name,n_fil,m,side", [("1", 1, 32, 64), ("2", 256, 64, 256), ("3", 4096, 32, 512),
                                               ("4a", 157, 64, 256), ("4b", 1563, 64, 640),
                                               ("4c", 15625, 64, 2048), ("5", 65536, 16, 2048)])
def test_config_shapes(name, n_fil, m, side):
    w = worlds.make_world(name)
    p = w["params"]
    assert (p["nx"], p["ny"]) == (side, side)
    assert len(w["offsets"]) == n_fil + 1 and int(w["offsets"][-1]) == n_fil * m == p["max_beads"]
    assert w["xy"].shape == (n_fil * m, 2) and w["xy"].dtype == np.float32
    for k in ("L_rest", "theta_rest", "k_bend", "k_shear", "k_stretch", "act_amp", "act_phase", "act_period"):
        assert w[k].shape == (n_fil * m,) and w[k].dtype == np.float32
    assert np.all(w["k_bend"] == 0.5) and np.all(w["act_period"] == np.float32(2.0))
    # initial shape = rest shape: unit edges
    xy = w["xy"].astype(np.float64).reshape(n_fil, m, 2)
    assert np.abs(np.linalg.norm(np.diff(xy, axis=1), axis=2) - 1.0).max() < 2e-3
    # travelling wave: joint amplitude 2 A sin(pi/(m-1)), zero at chain ends
    a = w["act_amp"].reshape(n_fil, m)
    assert np.all(a[:, 0] == 0) and np.all(a[:, -1] == 0)
    assert abs(a[0, 1] - 2 * 0.5 * math.sin(math.pi / (m - 1))) < 1e-6


def test_sweep_side_and_4d_size():
    assert [worlds.sweep_side(n) for n in (10_000, 100_000, 1_000_000, 10_000_000)] == [256, 640, 2048, 6272]
    assert worlds.SWEEP["4d"] == 10_000_000


def test_config3_has_static_source_and_config5_is_clustered():
    w3 = worlds.make_world("3")
    kinds = [f["kind"] for f in w3["params"]["fields"]]
    assert kinds == [0, 1] and w3["params"]["fields"][1]["sources"].shape == (1, 4)
    w5 = worlds.make_world("5")
    c = w5["xy"].reshape(-1, 16, 2).mean(axis=1)
    r = np.linalg.norm(c - 1024.0, axis=1)
    assert np.mean(r < 2.5 * 102.4) > 0.9  # Gaussian cluster, sigma = 5 % of the side


def test_ragged_world_translates_some_chains_by_whole_periods():
    w = worlds.ragged_world(96, 64, [3, 16, 33, 64], seed=1)
    assert list(w["offsets"]) == [0, 3, 19, 52, 116]
    assert w["xy"][:3, 0].max() < 0 or w["xy"][:3, 0].min() > 96  # chain 0 lives outside [0, nx)


def _joint_angles(w):
    """psi of every interior joint from the fp32 positions (plain numpy: input geometry only)."""
    off = w["offsets"]
    out = np.full(len(w["xy"]), np.nan)
    xy = w["xy"].astype(np.float64)
    for f in range(len(off) - 1):
        p = xy[off[f]:off[f + 1]]
        v = np.diff(p, axis=0)
        cr = v[:-1, 0] * v[1:, 1] - v[:-1, 1] * v[1:, 0]
        dt = (v[:-1] * v[1:]).sum(axis=1)
        out[off[f] + 1: off[f + 1] - 1] = np.arctan2(cr, dt)
    return out


def test_hairpin_world_holds_the_large_angle_cases():
    # the cases the GPU's K1 treats on its rare paths (k_filament.cuh half_kC / sin_small /
    # k_pack_params) must really be in the world the parity test runs
    w = worlds.hairpin_world()
    psi = _joint_angles(w)
    th = w["theta_rest"].astype(np.float64)
    inner = ~np.isnan(psi)
    assert np.any(np.abs(psi[inner] - math.pi) < 1e-3) and np.any(np.abs(psi[inner] + math.pi) < 1e-3)
    assert np.any(th > math.pi) and np.any(th < -math.pi) and np.any(th > 2 * math.pi)
    d = psi[inner] - th[inner]
    d = d - 2 * math.pi * np.round(d / (2 * math.pi))
    assert np.mean(np.abs(d) > 0.46) > 0.3        # beyond the small-angle atan range of K1
    assert np.mean(np.abs(psi[inner]) > 0.5 * math.pi) > 0.2   # dot <= 0: joints bent beyond 90 degrees
    # edges keep unit length (the hairpins fold the chain, they do not stretch it)
    off = w["offsets"]
    for f in range(len(off) - 1):
        v = np.diff(w["xy"][off[f]:off[f + 1]].astype(np.float64), axis=0)
        assert np.abs(np.linalg.norm(v, axis=1) - 1.0).max() < 1e-4

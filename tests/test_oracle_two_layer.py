"""Pins of the oracle's two-layer broadcast (mco_markers and the two_layer step; SURVEY 8(f)
NEXT-4, reading 28): "broadcasting the single filament into a two-layer version of
itself to artificially amplify a zero-thickness filament into a solid object"."""
import math

import numpy as np
import pytest

from oracle import mco
from paper_2607_02954_b200 import worlds

RNG = np.random.default_rng(31415)
CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])


def test_markers_of_a_straight_chain():
    a, h, m = 0.7, 0.5, 6
    t = np.array([math.cos(a), math.sin(a)])
    n = np.array([-t[1], t[0]])                       # tangent turned by +90 degrees
    xy = np.array([3.0, -2.0]) + np.arange(m)[:, None] * 1.1 * t
    M = mco.markers([0, m], xy, h)
    assert M.shape == (2 * m, 2)
    assert np.abs(M[0::2] - (xy + h * n)).max() < 1e-15     # entry 2i = X_i + h n_i
    assert np.abs(M[1::2] - (xy - h * n)).max() < 1e-15     # entry 2i+1 = X_i - h n_i


def test_markers_at_a_corner_and_at_the_ends():
    # right-angle corner: edge normals (0,1) and (-1,0) -> bead normal (-1,1)/sqrt 2; the end beads
    # take the normal of their only edge
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0]])
    M = mco.markers([0, 3], xy, 0.25)
    s = 0.25 / math.sqrt(2)
    want_plus = np.array([[0.0, 0.25], [1.0 - s, s], [0.75, 1.0]])
    assert np.abs(M[0::2] - want_plus).max() < 1e-15
    assert np.abs(0.5 * (M[0::2] + M[1::2]) - xy).max() < 1e-15      # the bead is the midpoint
    assert np.abs(np.linalg.norm(M[0::2] - M[1::2], axis=1) - 0.5).max() < 1e-15


def test_markers_are_frame_covariant_and_per_chain():
    lengths = [3, 7, 20]
    off = np.concatenate([[0], np.cumsum(lengths)]).astype(np.int32)
    xy = np.cumsum(RNG.normal(0, 1, (30, 2)), axis=0)
    th, sh = 2.2, np.array([5.0, 9.0])
    R = np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
    M = mco.markers(off, xy, 0.4)
    M2 = mco.markers(off, xy @ R.T + sh, 0.4)
    assert np.abs(M2 - (M @ R.T + sh)).max() < 1e-13
    # chains do not see each other: the last bead of chain 0 uses only its own edge
    v = xy[2] - xy[1]
    n = np.array([-v[1], v[0]]) / np.linalg.norm(v)
    assert np.abs(M[4] - (xy[2] + 0.4 * n)).max() < 1e-15
    # a hairpin whose two edge normals cancel falls back to the first edge's normal
    hp = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 0.0 + 0.0]])
    Mh = mco.markers([0, 3], hp, 0.3)
    assert np.abs(Mh[2] - np.array([1.0, 0.3])).max() < 1e-15


def _two_layer_world(h=0.5, **kw):
    w = worlds.ragged_world(64, 64, [5, 24, 33, 12], seed=29, static_source=True, **kw)
    w["params"] = dict(w["params"], two_layer=1, layer_offset=h)
    return w


def test_two_layer_step_glue_matches_components():
    # every grid exchange of the step goes through the markers with weight 1/2 each:
    # S2 deposit, S4 sampling, S5 spread, S7 interpolation -- rebuilt here from the pinned components
    w = _two_layer_world()
    p = w["params"]
    O = mco.World(w)
    O.set_state(3)
    X0 = w["xy"].astype(np.float64)
    O.step(1)
    s, it = O.read_state(), O.read_intermediates()
    nx, ny, N = p["nx"], p["ny"], len(X0)
    dt = float(np.float32(p["dt"]))
    M = mco.markers(w["offsets"], X0, 0.5)
    rho_b = 0.5 * mco.deposit(nx, ny, M)
    assert np.abs(it["rho_b"] - rho_b).max() < 1e-15
    assert abs(rho_b.sum() - N) < 1e-10                      # each bead still deposits unit mass
    f0 = p["fields"][0]
    R = mco.radius(f0["sigma"], f0["radius"])
    gx, gy = mco.grad(mco.blur(rho_b, float(np.float32(f0["sigma"])), R))
    pair = lambda a: 0.5 * (a[0::2] + a[1::2])
    F = float(np.float32(p["k_el"])) * dt * dt * it["D"]
    F = F - float(np.float32(f0["coupling"])) * dt * dt * pair(mco.interp(np.stack([gx, gy]), M))
    f1 = p["fields"][1]
    c = mco.static_field(nx, ny, f1["sources"])
    cgx, cgy = mco.grad(c)
    F = F + float(np.float32(f1["coupling"])) * dt * dt * pair(mco.interp(np.stack([cgx, cgy]), M))
    assert np.abs(s["force"] - F).max() < 1e-15
    assert np.abs(s["sense"] - pair(mco.interp(c[None], M))[:, 0]).max() < 1e-15
    G = mco.spread(nx, ny, M, np.repeat(0.5 * F, 2, axis=0))
    assert np.abs(it["G"] - G).max() < 1e-16
    assert np.abs(s["xy"] - (X0 + pair(mco.interp(s["u"], M)))).max() < 1e-13


def test_two_layer_conserves_force_and_power():
    w = _two_layer_world()
    O = mco.World(w)
    O.step(3)
    before = O.read_state()
    O.step(1)
    s, it = O.read_state(), O.read_intermediates()
    # total spread force unchanged by the doubling (each layer carries half)
    assert np.abs(it["G"].sum(axis=(1, 2)) - s["force"].sum(axis=0)).max() < 1e-13
    # power balance: S5 and S7 are adjoint with the SAME markers and weights,
    # sum_g G.u = sum_i F_i.U_i with U_i = this step's displacement
    U = s["xy"] - before["xy"]
    assert abs((it["G"] * s["u"]).sum() - (s["force"] * U).sum()) < 1e-12 * abs((s["force"] * U).sum()) + 1e-18
    # fluid momentum grows by the total bead force
    mom = lambda st: np.array([np.tensordot(CX, st["fdev"], 1).sum(), np.tensordot(CY, st["fdev"], 1).sum()])
    assert np.abs(mom(s) - mom(before) - s["force"].sum(axis=0)).max() < 1e-12


def test_two_layer_repulsion_is_pairwise_antisymmetric():
    # S4 samples with the adjoint of S2's deposit (same markers, same weights), so the steric
    # forces still sum to zero: no net self-propulsion from the repulsion field
    w = worlds.random_world(64, 64, 20, 12, seed=3, kappa=0.0, kappa_rep=0.05, clustered=4.0)
    w["params"] = dict(w["params"], two_layer=1, layer_offset=0.5)
    O = mco.World(w)
    O.step(1)
    F = O.read_state()["force"]
    assert np.abs(F).max() > 1e-5
    assert np.abs(F.sum(axis=0)).max() < 1e-15


def test_two_layer_tends_to_the_single_layer_as_h_vanishes():
    a = mco.World(_two_layer_world(h=1e-6))
    w1 = _two_layer_world()
    w1["params"] = dict(w1["params"], two_layer=0)
    b = mco.World(w1)
    for O in (a, b):
        O.step(5)
    sa, sb = a.read_state(), b.read_state()
    for k in ("xy", "u", "force"):
        assert np.linalg.norm(sa[k] - sb[k]) < 1e-5 * np.linalg.norm(sb[k]), k
    # ... and h = 1/2 is a different world: the force is spread over a wider band
    c = mco.World(_two_layer_world(h=0.5))
    c.step(5)
    assert np.linalg.norm(c.read_state()["u"] - sb["u"]) > 1e-3 * np.linalg.norm(sb["u"])


def test_two_layer_widens_the_band_of_a_straight_chain():
    # a straight horizontal chain pushed sideways: single layer spreads over 4 rows, two layers at
    # +-1/2 over 5 rows (amplified thickness), half of the force through each layer
    m = 16
    xy = np.stack([20.0 + np.arange(m), np.full(m, 30.0)], axis=1)
    F = np.tile([0.0, 1.0], (m, 1))
    G1 = mco.spread(64, 64, xy, F)
    M = mco.markers([0, m], xy, 0.5)
    Gp = mco.spread(64, 64, M[0::2], 0.5 * F)
    Gm = mco.spread(64, 64, M[1::2], 0.5 * F)
    assert abs(Gp[1].sum() - 0.5 * m) < 1e-12 and abs(Gm[1].sum() - 0.5 * m) < 1e-12
    rows = lambda G: int((np.abs(G[1]).sum(axis=1) > 1e-14).sum())
    assert rows(G1) == 3 and rows(Gp + Gm) == 5     # y = 30 is a node row: phi(+-2) = 0


def _pair_gram(M, nx, ny):
    """Gram matrix of the two-layer kernels: K_ij = sum_g delta2(g; i) delta2(g; j)."""
    n = len(M) // 2
    K = np.empty((n, n))
    for j in range(n):
        dj = 0.5 * mco.deposit(nx, ny, M[2 * j:2 * j + 2])
        s = mco.interp(dj[None], M)[:, 0]
        K[:, j] = 0.5 * (s[0::2] + s[1::2])
    return K


def test_mdf_through_one_layer_is_mco_mdf():
    nx, ny = 20, 24
    rng = np.random.default_rng(7)
    xy = np.stack([20 * worlds.uniform(1, "mdf-a", 30), 24 * worlds.uniform(1, "mdf-b", 30)], 1)
    V = 1e-2 * rng.standard_normal((30, 2))
    us = 1e-3 * rng.standard_normal((2, ny, nx))
    rho = 1 + 0.03 * rng.standard_normal((ny, nx))
    a, b = mco.mdf(xy, V, us, rho, 1.0, 4), mco.mdf_layers(xy, 1, V, us, rho, 1.0, 4)
    for k in ("F", "G", "u", "resid"):
        assert np.array_equal(a[k], b[k]), k


def test_two_layer_mdf_converges_to_the_no_slip_solution_of_a_dense_solve():
    # fixed point of the two-layer iteration: mean-over-markers interp(ustar + spread2(F)/(2 rho)) = V
    # <=> K F = 2 rho (V - Ustar), K the Gram matrix of the two-layer kernels; the error after k
    # iterations is (I - K/2)^k (F^0 - F_exact), exactly as for one layer (tests/test_oracle_mdf.py)
    nx, ny, rho = 24, 20, 1.05
    s = np.arange(9.0)
    xy = np.stack([6.3 + s * np.cos(0.4), 7.1 + s * np.sin(0.4)], 1)
    M = mco.markers([0, 9], xy, 0.5)
    rng = np.random.default_rng(4)
    V = 1e-2 * np.stack([np.cos(0.3 * s), 0.5 + np.sin(0.2 * s)], 1)
    us = 1e-4 * rng.standard_normal((2, ny, nx))
    K = _pair_gram(M, nx, ny)
    assert np.linalg.eigvalsh(K).max() < 4
    Um = mco.interp(us, M)
    Fex = np.linalg.solve(K, 2 * rho * (V - 0.5 * (Um[0::2] + Um[1::2])))
    for it in (1, 3, 32):
        r = mco.mdf_layers(M, 2, V, us, np.full((ny, nx), rho), rho, it)
        EK = np.linalg.matrix_power(np.eye(9) - 0.5 * K, it) @ (-Fex)
        assert np.allclose(r["F"] - Fex, EK, rtol=1e-9, atol=1e-15)
        assert np.allclose(r["G"].sum(axis=(1, 2)), r["F"].sum(axis=0), rtol=1e-12, atol=1e-18)
    assert np.all(np.diff(r["resid"]) < 0) and r["resid"][-1] < 0.1 * r["resid"][0]


def test_two_layer_mdf_step_glue_and_budgets():
    w = _two_layer_world(kappa_rep=0.01)
    w["params"] = dict(w["params"], coupling=1, mdf_iters=3)
    O = mco.World(w)
    O.step(2)
    before = O.read_state()
    O.step(1)
    s, it = O.read_state(), O.read_intermediates()
    X0 = before["xy"]
    M = mco.markers(w["offsets"], X0, 0.5)
    # the summed force and its grid image are those of the layered MDF on the step's own inputs
    f_pre = before["fdev"] + np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)[:, None, None]
    rho, ustar = mco.moments(f_pre)
    r1 = mco.mdf_layers(M, 2, np.zeros_like(X0), ustar, rho, 1.0, 1)      # V = 0: F = -rho0 * mean interp(u*)
    Um = mco.interp(ustar, M)
    assert np.allclose(r1["F"], -0.5 * (Um[0::2] + Um[1::2]), rtol=1e-13, atol=1e-18)
    assert np.allclose(it["G"].sum(axis=(1, 2)), s["force"].sum(axis=0), rtol=1e-11, atol=1e-16)
    U = s["xy"] - X0
    assert abs((it["G"] * s["u"]).sum() - (s["force"] * U).sum()) < 1e-11 * abs((s["force"] * U).sum()) + 1e-18
    mom = lambda st: np.array([np.tensordot(CX, st["fdev"], 1).sum(), np.tensordot(CY, st["fdev"], 1).sum()])
    assert np.abs(mom(s) - mom(before) - s["force"].sum(axis=0)).max() < 1e-12

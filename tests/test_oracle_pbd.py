"""Pins of the oracle's literal PBD (mco_pbd, reading 27): K
iterations of {bending pass Eq. 1, position pass Eq. 2-4}, Jacobi or red-black
Gauss-Seidel, rest length actuated like the rest angle, optional projection of the
advected positions."""
import math

import numpy as np
import pytest

from oracle import mco
from paper_2607_02954_b200 import worlds
from test_oracle_components import chain_arrays, chain_from_angles

RNG = np.random.default_rng(2718)
KEYS = ("L_rest", "theta_rest", "k_bend", "k_shear", "k_stretch", "act_amp", "act_phase", "act_period")


def run_pbd(xy, arrs, iters=1, order=0, dt=1e-2, n=0, offsets=None, act_L_amp=None):
    off = np.array([0, len(xy)], np.int32) if offsets is None else offsets
    return mco.pbd(off, xy, *[arrs[k] for k in KEYS], dt, n, iters, order, act_L_amp)


def random_chains(lengths, seed):
    rng = np.random.default_rng(seed)
    xs, arrs = [], {k: [] for k in KEYS}
    for m in lengths:
        th = rng.uniform(-0.6, 0.6, m)
        L = rng.uniform(0.8, 1.2, m)
        xy = chain_from_angles(th + rng.normal(0, 0.15, m), L * (1 + rng.normal(0, 0.05, m)),
                               x0=rng.uniform(-5, 40, 2), orient=rng.uniform(0, 6.28))
        xs.append(xy)
        a = chain_arrays(m, theta=th, kb=0.0, ks=0.0, kst=0.0, amp=0.0, phase=0.0, period=1.0)
        a["L_rest"] = L.astype(np.float32)
        for k in ("k_bend", "k_shear", "k_stretch"):
            a[k] = rng.uniform(0.2, 0.9, m).astype(np.float32)
        a["act_amp"] = rng.uniform(0, 0.2, m).astype(np.float32)
        a["act_phase"] = rng.uniform(0, 6.28, m).astype(np.float32)
        a["act_period"] = rng.uniform(0.5, 3.0, m).astype(np.float32)
        for k in KEYS:
            arrs[k].append(a[k])
    off = np.concatenate([[0], np.cumsum(lengths)]).astype(np.int32)
    return off, np.concatenate(xs), {k: np.concatenate(v) for k, v in arrs.items()}


def test_one_jacobi_iteration_is_mco_elastic_bit_for_bit():
    off, xy, arrs = random_chains([3, 4, 17, 64, 33], 1)
    for n in (0, 7, 123456):
        a = mco.elastic(off, xy, *[arrs[k] for k in KEYS], 1e-2, n)
        b = run_pbd(xy, arrs, iters=1, order=0, n=n, offsets=off)
        assert a.tobytes() == b.tobytes()


def test_jacobi_iterations_compose():
    # K iterations = K times {one iteration from the positions the previous ones produced}
    off, xy, arrs = random_chains([5, 40, 9], 2)
    Y, tot = xy.copy(), np.zeros_like(xy)
    for K in range(1, 6):
        tot = tot + mco.elastic(off, xy + tot, *[arrs[k] for k in KEYS], 1e-2, 11)
        D = run_pbd(xy, arrs, iters=K, order=0, n=11, offsets=off)
        assert np.abs(D - tot).max() < 1e-15
    assert np.abs(tot).max() > 1e-2   # the chains really are away from rest


def test_stretch_iterations_are_the_powers_of_the_jacobi_matrix():
    # collinear chain along its directors, k_bend irrelevant (all joint angles at rest): only Eq. 2
    # acts and one Jacobi iteration maps the edge excesses eps_e = l_e - L linearly,
    #   eps' = (I - k/2 T) eps,  T = tridiag(-1, 2, -1)   (x1 += dx, x2 -= dx on both neighbours),
    # so K iterations are the K-th matrix power: pins the iteration count and that every
    # correction of an iteration is computed from the same state.
    m, k, L = 12, 0.625, 1.0   # stiffnesses are stored as fp32: exactly representable values
    eps0 = RNG.uniform(-0.2, 0.2, m - 1)
    t = np.array([math.cos(0.7), math.sin(0.7)])
    s = np.concatenate([[0], np.cumsum(L + eps0)])
    xy = s[:, None] * t[None, :]
    arrs = chain_arrays(m, L=L, kst=k, ks=0.875, kb=0.5)
    T = 2 * np.eye(m - 1) - np.eye(m - 1, k=1) - np.eye(m - 1, k=-1)
    A = np.eye(m - 1) - 0.5 * k * T
    for K in (1, 2, 3, 8):
        D = run_pbd(xy, arrs, iters=K)
        new = xy + D
        lens = np.linalg.norm(np.diff(new, axis=0), axis=1)
        assert np.abs((lens - L) - np.linalg.matrix_power(A, K) @ eps0).max() < 1e-14
        v = np.diff(new, axis=0)
        assert np.abs(v[:, 0] * t[1] - v[:, 1] * t[0]).max() < 1e-14   # stays collinear


def test_gauss_seidel_sweep_by_hand():
    # red-black order on a collinear chain (pure stretch): even edges first, then the odd edges see
    # the moved beads.  4 beads, edges 0, 1, 2 with excesses e0, e1, e2 and stiffness k:
    #   d0 = k/2 e0, d2 = k/2 e2 (even edges, from the old positions)
    #   edge 1 then has excess e1 + d0 + d2 (bead 1 went back by d0, bead 2 forward by d2)
    #   d1 = k/2 (e1 + d0 + d2);  D = [d0, d1 - d0, d2 - d1, -d2] along t
    k, L = 0.75, 1.0            # fp32-exact
    e0, e1, e2 = 0.11, -0.07, 0.19
    t = np.array([math.cos(-1.1), math.sin(-1.1)])
    s = np.concatenate([[0], np.cumsum([L + e0, L + e1, L + e2])])
    xy = 3.0 + s[:, None] * t[None, :]
    arrs = chain_arrays(4, L=L, kst=k, ks=0.25, kb=0.375)
    D = run_pbd(xy, arrs, iters=1, order=1)
    d0, d2 = 0.5 * k * e0, 0.5 * k * e2
    d1 = 0.5 * k * (e1 + d0 + d2)
    want = np.array([d0, d1 - d0, d2 - d1, -d2])[:, None] * t[None, :]
    assert np.abs(D - want).max() < 1e-15
    # ... which differs from the Jacobi result (d1 = k/2 e1) by k/2 (d0 + d2) on the middle beads
    Dj = run_pbd(xy, arrs, iters=1, order=0)
    assert abs(np.linalg.norm(D[1] - Dj[1]) - 0.5 * k * (d0 + d2)) < 1e-15
    # 3 beads: even edge 0, then odd edge 1 with excess e1 + d0
    xy3 = xy[:3]
    D3 = run_pbd(xy3, chain_arrays(3, L=L, kst=k, ks=0.25, kb=0.375), iters=1, order=1)
    d1 = 0.5 * k * (e1 + d0)
    assert np.abs(D3 - np.array([d0, d1 - d0, -d1])[:, None] * t[None, :]).max() < 1e-15


def test_gauss_seidel_uses_the_directors_of_the_bending_pass():
    # 3-bead chain bent away from rest, |v| = L: edge 0 (even) is corrected first with the director
    # Rot(+k_b c/2) t_0; edge 1 (odd) then sees bead 1 moved by -dx_0 and keeps the director
    # Rot(-k_b c/2) t_1 formed from the ORIGINAL tangent (the bending pass precedes the position pass).
    kb, ks, kst, L, c = 0.5, 0.75, 0.625, 1.0, 0.2   # fp32-exact stiffnesses
    t0 = np.array([1.0, 0.0])
    t1 = np.array([math.cos(c), math.sin(c)])
    xy = np.array([[0, 0], L * t0, L * t0 + L * t1])
    arrs = chain_arrays(3, L=L, kb=kb, ks=ks, kst=kst)
    D = run_pbd(xy, arrs, iters=1, order=1)
    rot = lambda a, v: np.array([math.cos(a) * v[0] - math.sin(a) * v[1], math.sin(a) * v[0] + math.cos(a) * v[1]])
    d0, d1 = rot(0.5 * kb * c, t0), rot(-0.5 * kb * c, t1)
    dx0 = 0.5 * kst * ks * L * (t0 - d0)                     # |v_0| = L: no stretch part
    v1 = (xy[2]) - (xy[1] - dx0)                              # bead 1 moved by -dx_0
    l1 = np.linalg.norm(v1)
    cs = (l1 - L) * v1 / l1
    dx1 = 0.5 * kst * (cs + ks * (v1 - L * d1 - cs))
    assert np.abs(D - np.array([dx0, dx1 - dx0, -dx1])).max() < 1e-15


@pytest.mark.parametrize("order", [0, 1])
def test_net_displacement_sums_to_zero_and_is_frame_covariant(order):
    off, xy, arrs = random_chains([3, 8, 31, 64, 100], 5)
    la = RNG.uniform(0, 0.1, len(xy)).astype(np.float32)
    th, sh = 0.9, np.array([13.0, -40.0])
    R = np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
    for K in (1, 2, 4, 8):
        D = run_pbd(xy, arrs, iters=K, order=order, n=37, offsets=off, act_L_amp=la)
        for f in range(len(off) - 1):
            assert np.abs(D[off[f]:off[f + 1]].sum(axis=0)).max() < 1e-14     # Eq. 4 is symmetric
        D2 = run_pbd(xy @ R.T + sh, arrs, iters=K, order=order, n=37, offsets=off, act_L_amp=la)
        assert np.abs(D2 - D @ R.T).max() < 1e-13


@pytest.mark.parametrize("order", [0, 1])
def test_rest_shape_stays_at_rest_for_every_iteration_count(order):
    m = 30
    theta = RNG.uniform(-0.8, 0.8, m).astype(np.float32)
    L = RNG.uniform(0.7, 1.3, m).astype(np.float32)
    xy = chain_from_angles(theta.astype(float), L.astype(float), x0=(1.0, 2.0), orient=0.4)
    arrs = chain_arrays(m, theta=theta)
    arrs["L_rest"] = L
    assert np.abs(run_pbd(xy, arrs, iters=8, order=order, act_L_amp=np.zeros(m, np.float32))).max() < 1e-13


def test_rest_length_actuation_closed_form():
    # 3-bead collinear chain along its directors: dx_e = 1/2 k_st (l_e - L*_e(n)) t,
    # L*_e(n) = L_rest[e] + b_e sin(2 pi n dt / T_e + phi_e) with the period and phase of entry e
    L0, kst, dt, n = 1.0, 0.625, 1e-2, 57
    b = np.array([0.15, -0.08, 0.0], np.float32)
    T = np.array([1.3, 0.9, 1.0], np.float32)
    ph = np.array([0.4, 2.0, 0.0], np.float32)
    l = np.array([1.03, 0.96])
    t = np.array([math.cos(2.2), math.sin(2.2)])
    xy = np.concatenate([[0], np.cumsum(l)])[:, None] * t[None, :]
    arrs = chain_arrays(3, L=L0, kst=kst, ks=0.5, kb=0.0)
    arrs["act_period"], arrs["act_phase"] = T, ph
    D = run_pbd(xy, arrs, n=n, dt=dt, act_L_amp=b)
    Ls = L0 + b.astype(float) * np.sin(2 * math.pi * n * dt / T.astype(float) + ph.astype(float))
    d = 0.5 * kst * (l - Ls[:2])
    want = np.array([d[0], d[1] - d[0], -d[1]])[:, None] * t[None, :]
    assert np.abs(D - want).max() < 1e-15
    # no amplitude array = amplitude zero = the unactuated result
    assert run_pbd(xy, arrs, n=n, dt=dt).tobytes() == run_pbd(xy, arrs, n=n, dt=dt, act_L_amp=np.zeros(3, np.float32)).tobytes()
    # the rest ANGLE of entry e is driven by the same sine as the rest LENGTH of entry e
    arrs4 = chain_arrays(4, L=L0, kst=0.0, ks=0.0, kb=0.5, amp=0.3)
    arrs4["act_period"], arrs4["act_phase"] = np.full(4, 1.7, np.float32), np.full(4, 0.6, np.float32)
    s = math.sin(2 * math.pi * n * dt / float(np.float32(1.7)) + float(np.float32(0.6)))
    assert abs(s) > 0.3


@pytest.mark.parametrize("order", [0, 1])
def test_world_step_uses_the_iterated_pbd_and_projection(order):
    # glue: the world's D is mco_pbd of its parameters; with pbd_project the advected positions
    # receive the PBD displacement of the same step's targets once more
    w = worlds.ragged_world(64, 64, [5, 20, 33], seed=19)
    la = (0.05 * RNG.uniform(-1, 1, len(w["xy"]))).astype(np.float32)
    w["act_L_amp"] = la
    base = dict(w["params"], pbd_iters=3, pbd_order=order)
    A = mco.World(dict(w, params=dict(base, pbd_project=0)))
    B = mco.World(dict(w, params=dict(base, pbd_project=1)))
    for O in (A, B):
        O.set_state(4)
        O.step(1)
    a, b = A.read_state(), B.read_state()
    D = mco.pbd(w["offsets"], w["xy"].astype(np.float64), *[w[k] for k in KEYS], float(np.float32(base["dt"])), 4,
                3, order, la)
    assert np.abs(A.read_intermediates()["D"] - D).max() < 1e-16
    assert np.abs(a["u"] - b["u"]).max() == 0.0                  # the projection acts after S7
    Dp = mco.pbd(w["offsets"], a["xy"], *[w[k] for k in KEYS], float(np.float32(base["dt"])), 4, 3, order, la)
    assert np.abs(b["xy"] - (a["xy"] + Dp)).max() < 1e-13
    assert np.abs(Dp).max() > 1e-6

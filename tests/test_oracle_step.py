"""Pins of the oracle's whole step: the glue between the (separately pinned) components,
conservation laws of the coupled system, and the paper's physics claim (scallop theorem,
P:L57, L139, L155).  Absolute trajectories are "parity unpinned" (nothing in the paper
fixes them); see DESIGN.md.
"""
import math

import numpy as np
import pytest

from oracle import mco
from paper_2607_02954_b200 import worlds

CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])


def momentum(fdev):
    return np.array([np.tensordot(CX, fdev, 1).sum(), np.tensordot(CY, fdev, 1).sum()])


def test_empty_world_stays_at_rest():
    w = worlds.random_world(32, 32, 0, 8, seed=1)
    W = mco.World(w)
    W.step(3)
    s = W.read_state()
    assert s["step"] == 3
    assert np.abs(s["fdev"]).max() < 1e-15 and np.abs(s["u"]).max() < 1e-15
    assert np.allclose(s["rho"], 1.0, atol=1e-15)


def test_rest_shape_without_actuation_or_repulsion_does_not_move():
    w = worlds.random_world(48, 32, 5, 12, seed=2, kappa_rep=None)
    w["act_amp"][:] = 0
    W = mco.World(w)
    W.step(4)
    s = W.read_state()
    # the float32-rounded initial shape differs from the exact rest shape by ~ulp(X) ~ 4e-6,
    # so "zero" here is that size (the exact zero is pinned in test_oracle_components)
    assert np.abs(s["force"]).max() < 2e-5
    assert np.abs(s["xy"] - w["xy"].astype(np.float64)).max() < 2e-5
    assert np.abs(s["u"]).max() < 2e-5


def test_one_step_glue_matches_components():
    # couplings (kappa = k_el dt^2, kappa_rep = k_rep dt^2, kappa_chi = chi dt^2), signs
    # (-grad rho repels, +grad c attracts), order (same X for S1-S7, n before increment).
    w = worlds.random_world(32, 48, 6, 10, seed=3, static_source=True)
    # perturb away from rest so that every term is alive
    w["xy"] += (0.1 * worlds.normal(5, "pert", w["xy"].size).reshape(-1, 2)).astype(np.float32)
    p = w["params"]
    nx, ny, dt = p["nx"], p["ny"], np.float32(p["dt"]).astype(np.float64)
    W = mco.World(w)
    W.set_state(41)
    W.step(1)
    s, it = W.read_state(), W.read_intermediates()
    X0 = w["xy"].astype(np.float64)
    D = mco.elastic(w["offsets"], X0, w["L_rest"], w["theta_rest"], w["k_bend"], w["k_shear"],
                    w["k_stretch"], w["act_amp"], w["act_phase"], w["act_period"], dt, 41)
    assert np.array_equal(it["D"], D)
    k_el, k_rep, chi = (np.float64(np.float32(v)) for v in
                        (p["k_el"], p["fields"][0]["coupling"], p["fields"][1]["coupling"]))
    rho_b = mco.deposit(nx, ny, X0)
    rt = mco.blur(rho_b, 1.0, 5)
    c = mco.static_field(nx, ny, p["fields"][1]["sources"])
    F = k_el * dt * dt * D - k_rep * dt * dt * mco.interp(np.stack(mco.grad(rt)), X0) \
        + chi * dt * dt * mco.interp(np.stack(mco.grad(c)), X0)
    assert np.allclose(s["force"], F, rtol=1e-13, atol=1e-16)
    assert np.allclose(s["field"][0], rt, atol=1e-16) and np.allclose(s["field"][1], c, atol=1e-16)
    assert np.allclose(s["sense"], mco.interp(c[None], X0)[:, 0], atol=1e-15)
    G = mco.spread(nx, ny, X0, s["force"])
    assert np.allclose(it["G"], G, atol=1e-18)
    # first step from rest: rho = rho0, so u = G/2 exactly, and momentum after = sum F
    assert np.allclose(s["u"], 0.5 * G, atol=1e-17)
    assert np.allclose(momentum(s["fdev"]), s["force"].sum(axis=0), atol=1e-14)
    assert np.allclose(s["xy"], X0 + mco.interp(s["u"], X0), atol=1e-15)
    assert s["step"] == 42
    # chemotaxis sign: the chemical force points up the gradient of c
    gc = mco.interp(np.stack(mco.grad(c)), X0)
    W2 = mco.World(dict(w, params=dict(p, k_el=0.0, fields=[p["fields"][1]])))
    W2.step(1)
    assert np.all((W2.read_state()["force"] * gc).sum(axis=1) >= 0)


def test_total_momentum_only_changes_by_external_field_force():
    # elastic and repulsion forces are internal (sum to zero): fluid momentum stays ~0.
    w = worlds.random_world(32, 32, 8, 16, seed=4)
    W = mco.World(w)
    W.step(30)
    s = W.read_state()
    assert np.abs(s["force"]).max() > 1e-6
    assert np.abs(momentum(s["fdev"])).max() < 1e-14
    assert abs(s["fdev"].sum()) < 1e-11          # mass


def test_fp32_state_rounds_state_only():
    w = worlds.random_world(32, 32, 3, 16, seed=6)
    a, b = mco.World(w), mco.World(w, fp32_state=True)
    a.step(1)
    b.step(1)
    sa, sb = a.read_state(), b.read_state()
    assert np.array_equal(sb["xy"], sa["xy"].astype(np.float32).astype(np.float64))
    assert np.array_equal(sb["fdev"], sa["fdev"].astype(np.float32).astype(np.float64))
    assert np.array_equal(sb["u"], sa["u"])


def test_threads_do_not_change_results():
    w = worlds.random_world(32, 32, 6, 16, seed=7, static_source=True)
    a, b = mco.World(w), mco.World(w)
    a.step(5)
    b.set_threads(4)
    b.step(5)
    b.set_threads(0)
    sa, sb = a.read_state(), b.read_state()
    for k in ("xy", "u", "fdev", "force", "field", "sense"):
        assert np.array_equal(sa[k], sb[k]), k


def test_load_validation():
    w = worlds.random_world(32, 32, 2, 8, seed=8)
    bad = dict(w, k_bend=w["k_bend"] * 3)
    with pytest.raises(ValueError):
        mco.World(bad)
    bad = dict(w, offsets=np.array([0, 2, 16], np.int32))
    with pytest.raises(ValueError):
        mco.World(bad)
    for key, val in (("pbd_iters", 0), ("pbd_iters", 9), ("pbd_order", 2), ("pbd_project", 3),
                     ("two_layer", 2), ("layer_offset", 1.5)):
        bad = dict(w, params=dict(w["params"], **{key: val}))
        with pytest.raises(ValueError):
            mco.World(bad)
    mco.World(dict(w, params=dict(w["params"], pbd_iters=2, pbd_order=1))).close()


# ------------------------------------------------------------------ scallop theorem
def swimmer(nu_lat, kappa, kind):
    """32-bead straight chain on a 64^2 grid (config 1 geometry, no repulsion)."""
    w = worlds.make_world("1")
    p = w["params"]
    dt = p["dt"]
    p["nu"] = nu_lat / dt
    p["k_el"] = kappa / dt ** 2
    p["fields"] = []
    if kind == "hinge":                  # reciprocal: a single time-dependent angle
        w["act_amp"][:] = 0
        w["act_phase"][:] = 0
        w["act_amp"][10] = 0.5
    return w


def net_displacement_per_cycle(w, periods=10, steps_per=200):
    W = mco.World(w)
    W.step(steps_per * (periods // 2))
    c0 = W.read_state()["xy"].mean(axis=0)
    W.step(steps_per * (periods - periods // 2))
    c1 = W.read_state()["xy"].mean(axis=0)
    return (c1 - c0) / (periods - periods // 2)


def test_scallop_theorem_and_wave_direction():
    # "time-reversible strategies ... produce zero net displacement at high
    # viscosity, while non-reciprocal strategies ... maintain viable locomotion".
    ratios = []
    for nu_lat in (0.1, 0.5):
        wave = net_displacement_per_cycle(swimmer(nu_lat, 8.0, "wave"))
        hinge = net_displacement_per_cycle(swimmer(nu_lat, 8.0, "hinge"))
        ratios.append(np.linalg.norm(hinge) / np.linalg.norm(wave))
        # the phase -2 pi i/(m-1) makes the wave travel towards +i (+x); the swimmer moves -x
        assert wave[0] < 0 and abs(wave[0]) > 3 * abs(wave[1])
        assert np.linalg.norm(wave) > 5e-4
    assert ratios[0] < 0.25 and ratios[1] < 0.25
    assert ratios[1] < ratios[0]          # more viscous -> closer to zero


def test_viscosity_sweep_of_the_scallop_pair():
    # P:L151 "Viscosity is swept from 1e-3 to 2; this spans approximately Reynolds number Re ~ 1e3
    # to 1 ..., covering the transition from inertia-dominated to viscosity-dominated swimming";
    # P:L139 "time-reversible strategies ... produce zero net displacement at high viscosity";
    # P:L155 "Ultimately, a very high viscosity brings all movement close to a stop".
    # nu_lat over the paper's range, reciprocal single hinge against the travelling wave; the coupling
    # kappa is 2 in the thin-fluid half (stability limit of the stiff IBM spring) and 8 in
    # the viscous half, the two halves sharing nu_lat = 0.1.
    def pair(nu, kappa):
        h = np.linalg.norm(net_displacement_per_cycle(swimmer(nu, kappa, "hinge"), periods=6))
        wv = np.linalg.norm(net_displacement_per_cycle(swimmer(nu, kappa, "wave"), periods=6))
        return h, wv
    thin = [pair(nu, 2.0) for nu in (1e-3, 1e-2, 0.1)]
    thick = [pair(nu, 8.0) for nu in (0.1, 0.5, 2.0)]
    r_thin = [h / wv for h, wv in thin]
    r_thick = [h / wv for h, wv in thick]
    # inertia-dominated end: the reciprocal stroke DOES swim, even better than the wave (Re ~ 1e3)
    assert r_thin[0] > 1.0
    # ... and loses its advantage monotonically as the fluid thickens
    assert r_thin[0] > r_thin[1] > r_thin[2] and r_thin[2] < 0.3
    # viscosity-dominated half: scallop theorem, ever more strictly
    assert all(r < 0.25 for r in r_thick) and r_thick[0] > r_thick[1] > r_thick[2]
    # the reciprocal swimmer's own displacement falls monotonically across each half of the sweep
    assert thin[0][0] > thin[1][0] > thin[2][0] and thick[0][0] > thick[1][0] > thick[2][0]
    # close to a stop at the thick end: the wave at nu_lat = 2 covers < 10 % of its distance at 0.1
    assert thick[2][1] < 0.1 * thick[0][1]


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    # the oracle is built with -fsanitize=address,undefined and steps a world with
    # every option on; any out-of-bounds access, use of freed memory or undefined arithmetic aborts.
    # (compute-sanitizer is closed on the GPU pool; the CUDA path's memory safety rests on parity over
    # ragged / periodic / crowded worlds and on bit-reproducibility.)
    import os
    import subprocess
    import sys
    src = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "oracle", "mco.cpp")
    drv = tmp_path / "drive.cpp"
    drv.write_text(r"""
#include "mco.h"
#include <cstdio>
#include <cmath>
#include <vector>
int main() {
  for (int variant = 0; variant < 3; ++variant) {
    mco_world_params p = {};
    p.nx = 64; p.ny = 32; p.dt = 1e-2f; p.nu = 10.f; p.trt_lambda = 0.25f; p.rho0 = 1.f; p.k_el = 2e4f;
    p.pbd_iters = variant == 0 ? 1 : 3; p.pbd_order = variant == 2; p.pbd_project = variant == 2;
    p.two_layer = variant >= 1; p.layer_offset = 0.5f; p.coupling = variant == 1; p.mdf_iters = 2;
    float src4[4] = {10.f, 20.f, 1.f, 6.f};
    p.n_fields = 2;
    p.fields[0].kind = MCO_FIELD_BEAD_DENSITY; p.fields[0].sigma = 1.f; p.fields[0].radius = 5; p.fields[0].coupling = 100.f;
    p.fields[1].kind = MCO_FIELD_STATIC_SOURCE; p.fields[1].coupling = 200.f; p.fields[1].n_sources = 1; p.fields[1].sources = src4;
    const int lens[4] = {3, 17, 40, 5};
    std::vector<int32_t> off = {0};
    for (int m : lens) off.push_back(off.back() + m);
    const int N = off.back();
    p.max_beads = N;
    std::vector<float> xy(2 * N), L(N, 1.f), th(N, 0.1f), k(N, 0.5f), amp(N, 0.05f), ph(N, 0.3f), T(N, 2.f), la(N, 0.03f);
    for (int f = 0; f < 4; ++f)
      for (int i = off[f]; i < off[f + 1]; ++i) { xy[2 * i] = 60.f + 0.9f * (i - off[f]) + 64.f * (f - 1); xy[2 * i + 1] = 5.f + 7.f * f + 0.3f * std::sin(0.7f * i); }
    mco_world* w = nullptr;
    if (mco_create(&p, &w) != MCO_OK) return 2;
    if (mco_load_filaments(w, 4, off.data(), xy.data(), L.data(), th.data(), k.data(), k.data(), k.data(), amp.data(), ph.data(), T.data()) != MCO_OK) return 3;
    mco_set_length_actuation(w, la.data());
    mco_set_threads(w, 2);
    if (mco_step(w, 4) != MCO_OK) return 4;
    std::vector<double> X(2 * N), u(2 * 64 * 32);
    long long st = 0;
    mco_read_state(w, (int64_t*)&st, X.data(), u.data(), nullptr, nullptr, nullptr, nullptr, nullptr);
    if (st != 4 || !std::isfinite(X[0])) return 5;
    mco_destroy(w);
  }
  std::puts("sanitized ok");
  return 0;
}
""")
    exe = tmp_path / "drive"
    inc = os.path.dirname(src)
    r = subprocess.run(["g++", "-std=c++17", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined",
                        "-fno-sanitize-recover=all", f"-I{inc}", str(drv), src, "-o", str(exe)], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1", OMP_NUM_THREADS="2")
    r = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and "sanitized ok" in r.stdout, (r.returncode, r.stdout[-500:], r.stderr[-3000:])

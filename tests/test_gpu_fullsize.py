"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

Configs 2, 3, 4a, 4b: the whole per-step protocol of test_gpu_parity.py (every output, element
by element, 1e-5) at several steps.  Configs 4c and 5 (4.2 M nodes, ~1 M beads): one parity
step after a spin-up.  Config 4d (39 M nodes, 10 M beads -- the world bench.py times, the only one whose population
planes exceed 2^31 bytes): (a) one whole parity step against the threaded oracle, every output,
when the host has the memory for it (~30 GB); (b) always: every output compared with the oracle's
stateless components on WINDOWS (exact, because every stage of the step is local) at the domain
corner (0,0), the far corner and an interior tile boundary, and on sampled whole chains;
(c) properties that hold at any size -- exact run-to-run reproducibility, conservation of fluid
mass and the momentum budget, low-Mach guard.
"""
import numpy as np
import pytest

from paper_2607_02954_b200 import worlds
from test_gpu_parity import TOL_STEP, assert_close, assert_displacement, rel_l2, run_protocol

pytestmark = pytest.mark.gpu

CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1], dtype=np.float64)
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1], dtype=np.float64)


@pytest.mark.parametrize("name,steps_at", [("2", [0, 1, 10, 100]), ("3", [0, 1, 50]),
                                           ("4a", [0, 10, 100]), ("4b", [0, 20])])
def test_per_step_parity_config(name, steps_at):
    import os
    w = worlds.make_world(name)
    worst = run_protocol(w, steps_at=steps_at, threads=os.cpu_count() or 1)
    print(name, {k: f"{v:.2e}" for k, v in worst.items()})


def test_per_step_parity_many_ragged_chains():
    # 400 chains of 3..150 beads (K1's overlapping-window mode across thousands of windows)
    import os
    lengths = (3 + (worlds.uniform(5, "ragged/len", 400) * 148).astype(int)).tolist()
    w = worlds.ragged_world(256, 192, lengths, seed=21, static_source=True)
    worst = run_protocol(w, steps_at=[0, 7, 30], threads=os.cpu_count() or 1)
    print("ragged400", {k: f"{v:.2e}" for k, v in worst.items()})


@pytest.mark.parametrize("name", ["4c", "5"])
def test_one_parity_step_large(name):
    import os
    w = worlds.make_world(name)
    worst = run_protocol(w, steps_at=[8], threads=os.cpu_count() or 1)
    print(name, {k: f"{v:.2e}" for k, v in worst.items()})


@pytest.mark.parametrize("name", ["2", "5"])
def test_trajectory_100_steps_config(name):
    import os
    from oracle import mco
    from paper_2607_02954_b200 import binding
    w = worlds.make_world(name)
    G, O = binding.World(w), mco.World(w, threads=os.cpu_count() or 1)
    G.step(100)
    O.step(100)
    g, o = G.read_state(keys=("xy", "u")), O.read_state()
    assert_close("X after 100 steps", g["xy"], o["xy"], 1e-3)
    assert np.abs(o["u"]).max() < 0.1  # low-Mach guard of the input recipe


def _window(a, j0, i0, h, w):
    """Periodic window a[..., j0:j0+h, i0:i0+w] of a [.., ny, nx] array."""
    ny, nx = a.shape[-2:]
    jj = (np.arange(j0, j0 + h) % ny)[:, None]
    ii = (np.arange(i0, i0 + w) % nx)[None, :]
    return a[..., jj, ii]


W4D = 96          # window side (3 tiles); compared region = the window minus a margin
W4D_MARGIN = 16   # >= R + 1 + 2 (filter halo + gradient + bead support)


def _config_4d_windows(w, s0, s1, it, step0):
    """(b) element-wise comparison on windows: the oracle's component functions applied to the
    GPU's pre-step state cut out around the window; every stage is local, so the interior of the
    window is exactly what a whole-grid oracle step would give there."""
    from oracle import mco
    p = w["params"]
    nx, ny = p["nx"], p["ny"]
    dt = np.float64(np.float32(p["dt"]))
    kappa = np.float64(np.float32(p["k_el"])) * dt * dt
    fld = p["fields"][0]
    k_rep = np.float64(np.float32(fld["coupling"])) * dt * dt
    R = mco.radius(fld["sigma"], fld["radius"])
    op, om = mco.lattice_constants(np.float64(np.float32(p["nu"])), dt, np.float64(np.float32(p["trt_lambda"])))
    X0 = s0["xy"].astype(np.float64)
    off = w["offsets"]
    first = X0[off[:-1]]                                # first bead of every chain
    worst = {}
    M, Wn = W4D_MARGIN, W4D
    for (j0, i0) in ((-M, -M), (ny - Wn + M, nx - Wn + M), ((ny // 64) * 32 - 40, (nx // 96) * 32 - 40)):
        # beads whose support can touch the window: gather by CHAIN (elastic needs whole chains):
        # a 64-bead chain reaches at most 63 nodes from its first bead
        cx = (first[:, 0] - (i0 + Wn / 2)) % nx
        cy = (first[:, 1] - (j0 + Wn / 2)) % ny
        cx = np.minimum(cx, nx - cx)
        cy = np.minimum(cy, ny - cy)
        chains = np.nonzero((cx < Wn / 2 + 70) & (cy < Wn / 2 + 70))[0]
        idx = np.concatenate([np.arange(off[c], off[c + 1]) for c in chains])
        offs = np.concatenate([[0], np.cumsum(off[chains + 1] - off[chains])]).astype(np.int32)
        # local coordinates: window origin -> (0,0) of a periodic patch (Wn x Wn); beads outside
        # the patch wrap onto it and pollute only its margin... so use a patch big enough to hold
        # every gathered chain with room to spare: P = Wn + 2*160
        Pn = Wn + 320
        sh = np.array([i0 - 160, j0 - 160], dtype=np.float64)
        Xl = X0[idx] - sh
        Xl[:, 0] -= nx * np.round((Xl[:, 0] - Pn / 2) / nx)   # nearest periodic image to the patch
        Xl[:, 1] -= ny * np.round((Xl[:, 1] - Pn / 2) / ny)
        assert Xl.min() > 2 and Xl.max() < Pn - 3
        # S2 deposit, S3 filter + gradient on the patch (valid away from where other chains are missing:
        # chains whose first bead is > 70 + Wn/2 away cannot reach within 7 nodes of the window)
        rho_b = mco.deposit(Pn, Pn, Xl)
        blur = mco.blur(rho_b, float(fld["sigma"]), R)
        gx, gy = mco.grad(blur)
        sl = (slice(160 + M, 160 + Wn - M), slice(160 + M, 160 + Wn - M))       # compared region (patch coords)
        cj, ci = j0 + M, i0 + M
        h = Wn - 2 * M
        for name, gpu_a, orc_a in (("rho_b", _window(it["rho_b"], cj, ci, h, h), rho_b[sl]),
                                   ("field", _window(s1["field"][0], cj, ci, h, h), blur[sl])):
            worst[name] = max(worst.get(name, 0), assert_close(f"4d window {name}", gpu_a, orc_a))
        # S1 + S4 on the chains whose beads lie in the compared region
        D = mco.elastic(offs, Xl, *[w[k][idx] for k in ("L_rest", "theta_rest", "k_bend", "k_shear", "k_stretch",
                                                        "act_amp", "act_phase", "act_period")], dt, step0)
        Fo = kappa * D - k_rep * mco.interp(np.stack([gx, gy]), Xl)
        inside = ((Xl[:, 0] > 160 + M + 2) & (Xl[:, 0] < 160 + Wn - M - 3) &
                  (Xl[:, 1] > 160 + M + 2) & (Xl[:, 1] < 160 + Wn - M - 3))
        assert inside.sum() > 200
        worst["force"] = max(worst.get("force", 0), assert_close("4d window force", s1["force"][idx][inside], Fo[inside]))
        # S5 spread of the GPU's own forces
        Go = mco.spread(Pn, Pn, Xl, s1["force"][idx].astype(np.float64))
        worst["G"] = max(worst.get("G", 0), assert_close("4d window G", _window(it["G"], cj, ci, h, h), Go[(slice(None),) + sl]))
        # S6 on the patch of the GPU's pre-step populations and the GPU's G (periodic patch: valid
        # away from its rim)
        fpatch = _window(s0["fdev"], j0, i0, Wn, Wn).astype(np.float64) + \
            np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)[:, None, None] * np.float64(np.float32(p["rho0"]))
        Gpatch = _window(it["G"], j0, i0, Wn, Wn).astype(np.float64)
        f2, u = mco.lbm_step(fpatch, Gpatch, op, om)
        ins = (slice(M, Wn - M), slice(M, Wn - M))
        fdev2 = f2 - np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)[:, None, None] * np.float64(np.float32(p["rho0"]))
        for name, gpu_a, orc_a in (("u", _window(s1["u"], cj, ci, h, h), u[(slice(None),) + ins]),
                                   ("fdev", _window(s1["fdev"], cj, ci, h, h), fdev2[(slice(None),) + ins]),
                                   ("rho", _window(s1["rho"], cj, ci, h, h), f2.sum(axis=0)[ins])):
            worst[name] = max(worst.get(name, 0), assert_close(f"4d window {name}", gpu_a, orc_a))
        # S7 on the beads inside: the oracle's interpolation of the GPU's own u patch
        upatch = _window(s1["u"], j0 - 160 + 0, i0 - 160 + 0, Pn, Pn).astype(np.float64)
        U = mco.interp(upatch, Xl[inside])
        assert_displacement("4d window dX", s0["xy"][idx][inside], s1["xy"][idx][inside], U, rel=2e-6)
    return worst


def test_config_4d_against_the_oracle():
    import os
    from oracle import mco
    from paper_2607_02954_b200 import binding
    w = worlds.make_world("4d")
    p = w["params"]
    nx, ny = p["nx"], p["ny"]
    G = binding.World(w)
    G.keep_intermediates(True)
    G.step(5)
    s0 = G.read_state(keys=("xy", "fdev"))
    G.step(1)
    s1 = G.read_state()
    it = G.read_intermediates()
    G.close()
    # (c1) fluid mass is conserved exactly by collide+stream; momentum grows by sum(G)  (fp32 sums
    #     of 39 M terms: compare in fp64 with a tolerance scaled by the field's magnitude)
    m0 = s0["fdev"].astype(np.float64).sum()
    m1 = s1["fdev"].astype(np.float64).sum()
    assert abs(m1 - m0) < 1e-6 * np.abs(s1["fdev"]).astype(np.float64).sum()
    for C, ch in ((CX, 0), (CY, 1)):
        mom0 = np.tensordot(C, s0["fdev"].astype(np.float64).sum(axis=(1, 2)), 1)
        mom1 = np.tensordot(C, s1["fdev"].astype(np.float64).sum(axis=(1, 2)), 1)
        gsum = it["G"][ch].astype(np.float64).sum()
        assert abs((mom1 - mom0) - gsum) < 1e-5 * np.abs(it["G"][ch]).astype(np.float64).sum() + 1e-9
    # (c2) total spread force equals the sum of bead forces
    for ch in (0, 1):
        fs = s1["force"][:, ch].astype(np.float64).sum()
        gs = it["G"][ch].astype(np.float64).sum()
        assert abs(fs - gs) < 1e-5 * np.abs(s1["force"][:, ch]).astype(np.float64).sum()
    assert abs(it["rho_b"].astype(np.float64).sum() - len(s0["xy"])) < 1e-5 * len(s0["xy"])
    # (c3) low-Mach guard
    assert np.abs(s1["u"]).max() < 0.1 and np.abs(s1["rho"] - 1.0).max() < 0.1
    # (b) windows against the oracle's components
    worst = _config_4d_windows(w, s0, s1, it, 5)
    print("4d windows", {k: f"{v:.2e}" for k, v in worst.items()})
    # (a) the whole step against the threaded oracle, every output, when the host can hold it
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 0
    if avail < 40 * 2 ** 30:
        pytest.skip(f"windows compared; whole-grid oracle step skipped ({avail / 2**30:.0f} GiB of host memory free, ~30 needed)")
    O = mco.World(w, threads=os.cpu_count() or 1)
    O.set_state(s0["step"], xy=s0["xy"].astype(np.float64), fdev=s0["fdev"].astype(np.float64))
    O.step(1)
    o = O.read_state()
    oi = O.read_intermediates()
    O.close()
    full = {}
    for name, a, b in (("xy", s1["xy"], o["xy"]), ("u", s1["u"], o["u"]), ("rho", s1["rho"], o["rho"]),
                       ("fdev", s1["fdev"], o["fdev"]), ("force", s1["force"], o["force"]),
                       ("field", s1["field"], o["field"]), ("rho_b", it["rho_b"], oi["rho_b"]),
                       ("G", it["G"], oi["G"])):
        full[name] = assert_close(f"4d {name}", a, b)
    full["dX/bound"] = assert_displacement("4d dX vs oracle", s0["xy"], s1["xy"], o["xy"] - s0["xy"].astype(np.float64))
    print("4d whole step", {k: f"{v:.2e}" for k, v in full.items()})


def test_config_4d_bitwise_reproducible_and_keep_g_is_neutral():
    # run to run at full size, and the KEEP_G variant of the fused kernel (the one the parity tests
    # run) against the plain one (the one bench.py times)
    from paper_2607_02954_b200 import binding
    w = worlds.make_world("4d")
    outs = []
    for keep in (False, False, True):
        H = binding.World(w)
        H.keep_intermediates(keep)
        H.step(6)
        outs.append(H.read_state(keys=("xy", "u", "force")))
        H.close()
    for o in outs[1:]:
        for k in ("xy", "u", "force"):
            assert outs[0][k].tobytes() == o[k].tobytes(), k

"""Seeded synthetic worlds (inputs only -- none of the method's arithmetic lives here).

These are the input generators shared by the CUDA path and the CPU oracle (the only
thing the two share).  The recipe is DESIGN.md "Input recipe" / SURVEY.md 8(d): the
paper's scaling workload (many filaments on one fixed grid, hundreds to a
thousand steps) gives the shape; its unspecified creature content is replaced by
seeded random chains.  No dataset or benchmark suite is involved.

A world is a plain dict:
  params : dict of world parameters (python scalars; fields = list of dicts)
  offsets: int32 [n_fil+1]
  xy, L_rest, theta_rest, k_bend, k_shear, k_stretch, act_amp, act_phase, act_period:
           float32 arrays ([N,2] for xy, [N] otherwise), chain-ordered
  steps  : number of steps BASELINE.json asks for on this config
"""
from __future__ import annotations

import math

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return z ^ (z >> np.uint64(31))


def _stream_id(name: str) -> int:
    h = 1469598103934665603  # FNV-1a, version-proof
    for ch in name.encode():
        h = ((h ^ ch) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
    return h


def uniform(seed: int, stream: str, n: int) -> np.ndarray:
    """Counter-based uniform [0,1) with 24 bits, float64 array of length n."""
    with np.errstate(over="ignore"):
        base = _splitmix64(np.array([(seed * 0x632BE59BD9B4E019 + _stream_id(stream))
                                     & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))[0]
        k = np.arange(n, dtype=np.uint64)
        z = _splitmix64((base + k * np.uint64(0xD1342543DE82EF95)) & _M64)
    return (z >> np.uint64(40)).astype(np.float64) / float(1 << 24)


def normal(seed: int, stream: str, n: int) -> np.ndarray:
    u1 = uniform(seed, stream + "/u1", n)
    u2 = uniform(seed, stream + "/u2", n)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


def default_params(nx: int, ny: int, kappa: float, kappa_rep: float, *, dt: float = 1e-2,
                   nu: float = 10.0, sigma: float = 1.0, radius: int = 5) -> dict:
    """Lattice couplings kappa (= k_el dt^2) and kappa_rep (= k_rep dt^2) are converted
    to the physical inputs the ABI takes."""
    fields = []
    if kappa_rep is not None:
        fields.append(dict(kind=0, sigma=sigma, radius=radius, coupling=kappa_rep / dt ** 2,
                           sources=None))
    return dict(nx=nx, ny=ny, dt=dt, nu=nu, trt_lambda=0.25, rho0=1.0, k_el=kappa / dt ** 2,
                pbd_iters=1, fields=fields, max_beads=0)


def build_chains(theta0: np.ndarray, centres: np.ndarray, orient: np.ndarray,
                 psi: np.ndarray, *, L0: float = 1.0, k: float = 0.5, amp_tangent: float = 0.5,
                 period_steps: float = 200.0, dt: float = 1e-2) -> dict:
    """theta0 [n_fil, m] rest joint angles (columns 0 and m-1 ignored), centres [n_fil,2],
    orient [n_fil], psi [n_fil] -> chain arrays.  Initial shape = rest shape."""
    n_fil, m = theta0.shape
    th = theta0.astype(np.float64).copy()
    th[:, 0] = 0.0
    th[:, m - 1] = 0.0
    # tangent angle of edge e: alpha_0 = orientation, alpha_e = alpha_{e-1} + theta0_e
    alpha = orient[:, None] + np.cumsum(th[:, : m - 1], axis=1)  # th[:,0] == 0
    x = np.zeros((n_fil, m))
    y = np.zeros((n_fil, m))
    x[:, 1:] = np.cumsum(L0 * np.cos(alpha), axis=1)
    y[:, 1:] = np.cumsum(L0 * np.sin(alpha), axis=1)
    x += (centres[:, 0] - x.mean(axis=1))[:, None]
    y += (centres[:, 1] - y.mean(axis=1))[:, None]
    idx = np.arange(m, dtype=np.float64)[None, :]
    interior = np.zeros((1, m))
    interior[0, 1: m - 1] = 1.0
    a_joint = 2.0 * amp_tangent * math.sin(math.pi / (m - 1))
    amp = np.broadcast_to(a_joint * interior, (n_fil, m))
    phase = (psi[:, None] - 2.0 * math.pi * idx / (m - 1)) * interior
    N = n_fil * m
    f32 = np.float32
    return dict(
        offsets=(np.arange(n_fil + 1, dtype=np.int64) * m).astype(np.int32),
        xy=np.stack([x.reshape(N), y.reshape(N)], axis=1).astype(f32),
        L_rest=np.full(N, L0, f32),
        theta_rest=th.reshape(N).astype(f32),
        k_bend=np.full(N, k, f32), k_shear=np.full(N, k, f32), k_stretch=np.full(N, k, f32),
        act_amp=np.ascontiguousarray(amp).reshape(N).astype(f32),
        act_phase=phase.reshape(N).astype(f32),
        act_period=np.full(N, period_steps * dt, f32),
    )


def _random_chains(tag: str, seed: int, n_fil: int, m: int, nx: int, ny: int, *,
                   centres: np.ndarray | None = None, theta_lim: float = 0.3) -> dict:
    th = (uniform(seed, tag + "/theta0", n_fil * m).reshape(n_fil, m) * 2.0 - 1.0) * theta_lim
    if centres is None:
        centres = np.stack([uniform(seed, tag + "/cx", n_fil) * nx,
                            uniform(seed, tag + "/cy", n_fil) * ny], axis=1)
    orient = uniform(seed, tag + "/orient", n_fil) * 2.0 * math.pi
    psi = uniform(seed, tag + "/psi", n_fil) * 2.0 * math.pi
    return build_chains(th, centres, orient, psi)


def sweep_side(n_beads: int) -> int:
    return max(128, int(round(math.sqrt(4.0 * n_beads) / 128.0)) * 128)


SWEEP = {"4a": 10_000, "4b": 100_000, "4c": 1_000_000, "4d": 10_000_000}


def make_world(name: str, seed: int = 0) -> dict:
    """BASELINE.json configs: '1', '2', '3', '4a'..'4d', '5'."""
    if name == "1":
        nx = ny = 64
        m = 32
        w = build_chains(np.zeros((1, m)), np.array([[32.0, 32.0]]), np.zeros(1), np.zeros(1))
        params, steps = default_params(nx, ny, kappa=8.0, kappa_rep=0.01), 100
    elif name == "2":
        nx = ny = 256
        w = _random_chains("cfg2", seed, 256, 64, nx, ny)
        params, steps = default_params(nx, ny, kappa=2.0, kappa_rep=0.01), 1000
    elif name == "3":
        nx = ny = 512
        n_fil, m = 4096, 32
        cls = np.arange(n_fil) % 3
        big_theta = (uniform(seed, "cfg3/arc", n_fil) * 2.0 - 1.0) * math.pi
        zeta = 0.3 + 0.5 * uniform(seed, "cfg3/zig", n_fil)
        sign = np.where(np.arange(m) % 2 == 0, 1.0, -1.0)[None, :]
        th = np.zeros((n_fil, m))
        th = np.where((cls == 1)[:, None], (big_theta / (m - 2))[:, None], th)
        th = np.where((cls == 2)[:, None], zeta[:, None] * sign, th)
        centres = np.stack([uniform(seed, "cfg3/cx", n_fil) * nx,
                            uniform(seed, "cfg3/cy", n_fil) * ny], axis=1)
        orient = uniform(seed, "cfg3/orient", n_fil) * 2.0 * math.pi
        psi = uniform(seed, "cfg3/psi", n_fil) * 2.0 * math.pi
        w = build_chains(th, centres, orient, psi)
        params, steps = default_params(nx, ny, kappa=2.0, kappa_rep=0.01), 1000
        dt = params["dt"]
        params["fields"].append(dict(kind=1, sigma=0.0, radius=0, coupling=0.02 / dt ** 2,
                                     sources=np.array([[256.0, 256.0, 1.0, 51.2]], np.float32)))
    elif name in SWEEP:
        n = SWEEP[name]
        n_fil = -(-n // 64)
        nx = ny = sweep_side(n)
        w = _random_chains("cfg" + name, seed, n_fil, 64, nx, ny)
        params, steps = default_params(nx, ny, kappa=2.0, kappa_rep=0.01), 200
    elif name == "5":
        nx = ny = 2048
        n_fil, m = 65536, 16
        centres = np.stack([1024.0 + 102.4 * normal(seed, "cfg5/cx", n_fil),
                            1024.0 + 102.4 * normal(seed, "cfg5/cy", n_fil)], axis=1)
        w = _random_chains("cfg5", seed, n_fil, m, nx, ny, centres=centres)
        params, steps = default_params(nx, ny, kappa=0.25, kappa_rep=2e-4), 500
    else:
        raise ValueError(f"unknown world {name!r}")
    params["max_beads"] = int(w["offsets"][-1])
    w["params"] = params
    w["steps"] = steps
    w["name"] = name
    return w


def random_world(nx: int, ny: int, n_fil: int, m: int, seed: int = 0, *, kappa: float = 2.0,
                 kappa_rep: float | None = 0.01, nu: float = 10.0, static_source: bool = False,
                 clustered: float = 0.0, tag: str = "rw") -> dict:
    """Small worlds of the same recipe for parity tests (ragged tiles, wrap, both field
    kinds).  clustered > 0: Gaussian-clustered centres with that sigma (cells)."""
    centres = None
    if clustered > 0:
        centres = np.stack([nx / 2 + clustered * normal(seed, tag + "/ccx", n_fil),
                            ny / 2 + clustered * normal(seed, tag + "/ccy", n_fil)], axis=1)
    w = _random_chains(tag, seed, n_fil, m, nx, ny, centres=centres)
    params = default_params(nx, ny, kappa=kappa, kappa_rep=kappa_rep, nu=nu)
    if static_source:
        dt = params["dt"]
        params["fields"].append(dict(kind=1, sigma=0.0, radius=0, coupling=0.02 / dt ** 2,
                                     sources=np.array([[nx * 0.5, ny * 0.25, 1.0, nx * 0.1],
                                                       [nx * 0.1, ny * 0.9, 0.5, nx * 0.05]],
                                                      np.float32)))
    params["max_beads"] = int(w["offsets"][-1])
    w["params"] = params
    w["steps"] = 100
    w["name"] = tag
    return w


def ragged_world(nx: int, ny: int, lengths, seed: int = 0, *, kappa: float = 2.0,
                 kappa_rep: float | None = 0.01, static_source: bool = False,
                 shift_some: bool = True, tag: str = "rg") -> dict:
    """Chains of different lengths (edge cases of the one-warp-per-chain kernel: shorter than,
    equal to and longer than a warp), uniformly placed so that some straddle the periodic
    boundary; with shift_some every third chain is translated by a whole number of domain
    periods, so unwrapped coordinates well outside [0,nx) x [0,ny) are exercised."""
    parts = []
    for g, m in enumerate(lengths):
        parts.append(_random_chains(f"{tag}/{g}", seed, 1, int(m), nx, ny))
    keys = ("xy", "L_rest", "theta_rest", "k_bend", "k_shear", "k_stretch", "act_amp",
            "act_phase", "act_period")
    w = {k: np.concatenate([p[k] for p in parts], axis=0) for k in keys}
    w["offsets"] = np.concatenate([[0], np.cumsum([int(m) for m in lengths])]).astype(np.int32)
    if shift_some:
        for f in range(0, len(lengths), 3):
            s, e = w["offsets"][f], w["offsets"][f + 1]
            w["xy"][s:e, 0] += np.float32(nx * (1 if f % 2 else -2))
            w["xy"][s:e, 1] += np.float32(ny * (-1 if f % 2 else 1))
    base = random_world(nx, ny, 1, 4, seed=seed, kappa=kappa, kappa_rep=kappa_rep,
                        static_source=static_source, tag=tag + "/p")
    params = base["params"]
    params["max_beads"] = int(w["offsets"][-1])
    w["params"] = params
    w["steps"] = 100
    w["name"] = tag
    return w


def chains_from_angles(psi0: np.ndarray, theta_rest: np.ndarray, centres: np.ndarray,
                       orient: np.ndarray, phase0: np.ndarray, *, L0: float = 1.0, k: float = 0.5,
                       amp_tangent: float = 0.5, period_steps: float = 200.0, dt: float = 1e-2) -> dict:
    """Like build_chains, but the INITIAL joint angles psi0 [n_fil, m] and the rest angles
    theta_rest [n_fil, m] are given separately (columns 0 and m-1 ignored): chains that start
    away from their rest shape."""
    base = build_chains(psi0, centres, orient, phase0, L0=L0, k=k, amp_tangent=amp_tangent,
                        period_steps=period_steps, dt=dt)
    th = theta_rest.astype(np.float64).copy()
    th[:, 0] = 0.0
    th[:, -1] = 0.0
    base["theta_rest"] = th.reshape(-1).astype(np.float32)
    return base


def hairpin_world(nx: int = 96, ny: int = 64, n_fil: int = 24, m: int = 20, seed: int = 0, *,
                  kappa: float = 0.01, kappa_rep: float | None = 1e-4, tag: str = "hp") -> dict:
    """Chains far from rest, for the large-angle paths of the elastic operator (Eq. 1, P:L95-98;
    readings 4 and 25): rest angles ~U(-3, 3) rad, initial joint angles = rest angle + U(-1.5,
    1.5) wrapped to (-pi, pi], and in chain f (f = 0..5) one joint forced to a special case:
      f=0: psi = +pi - 5e-4 (hairpin, just inside the branch cut)   f=1: psi = -pi + 7e-4
      f=2: theta_rest = 3.5 > pi      f=3: theta_rest = -4.0 < -pi   f=4: theta_rest = 2 pi + 0.3
      f=5: psi = pi/2 exactly on the small-angle / large-angle boundary of a rest angle 0.
    The couplings are weak (kappa = 0.01) so that the O(1) displacements these joints ask for
    keep the fluid at low Mach number."""
    th = (uniform(seed, tag + "/theta", n_fil * m).reshape(n_fil, m) * 2.0 - 1.0) * 3.0
    pert = (uniform(seed, tag + "/pert", n_fil * m).reshape(n_fil, m) * 2.0 - 1.0) * 1.5
    psi = th + pert
    psi = psi - 2.0 * math.pi * np.round(psi / (2.0 * math.pi))   # into [-pi, pi]
    j = m // 2
    psi[0, j] = math.pi - 5e-4
    psi[1, j] = -math.pi + 7e-4
    th[2, j], th[3, j], th[4, j] = 3.5, -4.0, 2.0 * math.pi + 0.3
    th[5, j], psi[5, j] = 0.0, 0.5 * math.pi
    centres = np.stack([uniform(seed, tag + "/cx", n_fil) * nx, uniform(seed, tag + "/cy", n_fil) * ny], axis=1)
    orient = uniform(seed, tag + "/orient", n_fil) * 2.0 * math.pi
    ph = uniform(seed, tag + "/psi", n_fil) * 2.0 * math.pi
    w = chains_from_angles(psi, th, centres, orient, ph)
    params = default_params(nx, ny, kappa=kappa, kappa_rep=kappa_rep)
    params["max_beads"] = int(w["offsets"][-1])
    w["params"] = params
    w["steps"] = 20
    w["name"] = tag
    return w

"""Thin ctypes binding of libmc.so (include/mc.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used for device
memory (the workspace and the in/out arrays) and the stream.  There is no CPU fallback:
`load_library()` raises if libmc.so is missing and `World` raises without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmc.so")

MC_OK, MC_EINVAL, MC_ENOMEM, MC_ECUDA, MC_ESTATE, MC_EDIVERGED = 0, -1, -2, -3, -4, -5
SYMBOLS = ("mc_workspace_bytes", "mc_create", "mc_load_filaments", "mc_step", "mc_read_state",
           "mc_read_intermediates", "mc_launch_count", "mc_destroy", "mc_last_error",
           "mc_profile_enable", "mc_profile_read", "mc_keep_intermediates", "mc_texture_gathers",
           "mc_cluster_tiles", "mc_set_positions", "mc_set_length_actuation", "mc_load_fluid", "mc_batch_workspace_bytes",
           "mc_create_batch", "mc_load_filaments_batch", "mc_step_batch", "mc_batch_world", "mc_destroy_batch",
           "mc_batch_last_error", "mc_set_positions_batch", "mc_read_positions_batch", "mc_deposit_noalloc",
           "mc_noalloc_last_error")
NOALLOC_MAX_BEADS, NOALLOC_MAX_TILES = 32768, 1024
PROF_SLOTS = ("K0_bin", "K2a_deposit", "K3a_blur_grad", "K1_filament", "K2b_spread", "K3b_lbm",
              "K4_interp_integrate")

_fp = C.POINTER(C.c_float)


class FieldParams(C.Structure):
    _fields_ = [("kind", C.c_int32), ("sigma", C.c_float), ("radius", C.c_int32),
                ("coupling", C.c_float), ("n_sources", C.c_int32), ("sources", _fp)]


class WorldParams(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("dt", C.c_float), ("nu", C.c_float),
                ("trt_lambda", C.c_float), ("rho0", C.c_float), ("k_el", C.c_float),
                ("pbd_iters", C.c_int32), ("n_fields", C.c_int32), ("fields", FieldParams * 4),
                ("max_beads", C.c_int64), ("coupling", C.c_int32), ("mdf_iters", C.c_int32),
                ("pbd_order", C.c_int32), ("pbd_project", C.c_int32), ("two_layer", C.c_int32),
                ("layer_offset", C.c_float)]


class McError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libmc error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libmc.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2607_02954_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.mc_workspace_bytes.restype = C.c_size_t
    L.mc_workspace_bytes.argtypes = [C.POINTER(WorldParams)]
    L.mc_create.restype = C.c_int
    L.mc_create.argtypes = [C.POINTER(WorldParams), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.mc_load_filaments.restype = C.c_int
    L.mc_load_filaments.argtypes = [vp, i32, C.POINTER(i32)] + [vp] * 9
    L.mc_step.restype = C.c_int
    L.mc_step.argtypes = [vp, i32]
    L.mc_read_state.restype = C.c_int
    L.mc_read_state.argtypes = [vp, C.POINTER(i64)] + [vp] * 7
    L.mc_read_intermediates.restype = C.c_int
    L.mc_read_intermediates.argtypes = [vp, vp, vp]
    L.mc_launch_count.restype = i64
    L.mc_launch_count.argtypes = [vp]
    L.mc_profile_enable.restype = C.c_int
    L.mc_profile_enable.argtypes = [vp, i32]
    L.mc_profile_read.restype = C.c_int
    L.mc_profile_read.argtypes = [vp, _fp, C.POINTER(i32)]
    L.mc_keep_intermediates.restype = C.c_int
    L.mc_keep_intermediates.argtypes = [vp, i32]
    L.mc_texture_gathers.restype = C.c_int
    L.mc_texture_gathers.argtypes = [vp, i32]
    L.mc_set_positions.restype = C.c_int
    L.mc_set_positions.argtypes = [vp, vp]
    L.mc_cluster_tiles.restype = C.c_int
    L.mc_cluster_tiles.argtypes = [vp, i32]
    L.mc_load_fluid.restype = C.c_int
    L.mc_load_fluid.argtypes = [vp, i64, vp]
    L.mc_set_length_actuation.restype = C.c_int
    L.mc_set_length_actuation.argtypes = [vp, vp]
    L.mc_batch_workspace_bytes.restype = C.c_size_t
    L.mc_batch_workspace_bytes.argtypes = [C.POINTER(WorldParams), i32]
    L.mc_create_batch.restype = C.c_int
    L.mc_create_batch.argtypes = [C.POINTER(WorldParams), i32, vp, C.c_size_t, vp, C.POINTER(vp)]
    L.mc_load_filaments_batch.restype = C.c_int
    L.mc_load_filaments_batch.argtypes = [vp, i32, C.POINTER(i32)] + [vp] * 10
    L.mc_step_batch.restype = C.c_int
    L.mc_step_batch.argtypes = [vp, i32]
    L.mc_set_positions_batch.restype = C.c_int
    L.mc_set_positions_batch.argtypes = [vp, vp]
    L.mc_read_positions_batch.restype = C.c_int
    L.mc_read_positions_batch.argtypes = [vp, C.POINTER(i64), vp]
    L.mc_deposit_noalloc.restype = C.c_int
    L.mc_deposit_noalloc.argtypes = [i32, i32, i32, vp, vp, vp]
    L.mc_noalloc_last_error.restype = C.c_char_p
    L.mc_noalloc_last_error.argtypes = []
    L.mc_batch_world.restype = vp
    L.mc_batch_world.argtypes = [vp, i32]
    L.mc_destroy_batch.restype = None
    L.mc_destroy_batch.argtypes = [vp]
    L.mc_batch_last_error.restype = C.c_char_p
    L.mc_batch_last_error.argtypes = [vp]
    L.mc_destroy.restype = None
    L.mc_destroy.argtypes = [vp]
    L.mc_last_error.restype = C.c_char_p
    L.mc_last_error.argtypes = [vp]
    _lib = L
    return L


def make_params(p: dict):
    """worlds.py params dict -> (WorldParams, keepalive)."""
    wp = WorldParams()
    keep = []
    for k in ("nx", "ny", "pbd_iters"):
        setattr(wp, k, int(p[k]))
    for k in ("dt", "nu", "trt_lambda", "rho0", "k_el"):
        setattr(wp, k, float(p[k]))
    wp.n_fields = len(p["fields"])
    wp.max_beads = int(p["max_beads"])
    wp.coupling = int(p.get("coupling", 0))
    wp.mdf_iters = int(p.get("mdf_iters", 0))
    wp.pbd_order = int(p.get("pbd_order", 0))
    wp.pbd_project = int(p.get("pbd_project", 0))
    wp.two_layer = int(p.get("two_layer", 0))
    wp.layer_offset = float(p.get("layer_offset", 0.0))
    for i, fd in enumerate(p["fields"][:4]):
        fp = wp.fields[i]
        fp.kind, fp.sigma = int(fd["kind"]), float(fd["sigma"])
        fp.radius, fp.coupling = int(fd["radius"]), float(fd["coupling"])
        src = fd.get("sources")
        if src is not None:
            src = np.ascontiguousarray(src, dtype=np.float32).reshape(-1, 4)
            keep.append(src)
            fp.n_sources = src.shape[0]
            fp.sources = src.ctypes.data_as(_fp)
        else:
            fp.n_sources = 0
            fp.sources = None
    return wp, keep


def workspace_bytes(params: dict) -> int:
    wp, _keep = make_params(params)
    return int(load_library().mc_workspace_bytes(C.byref(wp)))


_CHAIN_KEYS = ("xy", "L_rest", "theta_rest", "k_bend", "k_shear", "k_stretch", "act_amp",
               "act_phase", "act_period")


class World:
    """mc_create + mc_load_filaments from a worlds.py dict; mc_step; mc_read_state."""

    def __init__(self, world: dict, device: str = "cuda:0", stream=None, _member=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2607_02954_b200 needs a CUDA device (no CPU fallback)")
        L = load_library()
        self.torch = torch
        self.device = torch.device(device)
        self.p = world["params"]
        self.nx, self.ny = int(self.p["nx"]), int(self.p["ny"])
        self.n_fields = len(self.p["fields"])
        self.h = None
        self.owned = _member is None
        if _member is not None:  # world k of a Batch: the batch owns the handle, the workspace and the stream
            self.h, self.stream, self.N = _member
            self.workspace = None
            return
        with torch.cuda.device(self.device):
            # a stream of its own: the legacy default stream cannot be captured into CUDA graphs
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            wp, keep = make_params(self.p)
            nbytes = int(L.mc_workspace_bytes(C.byref(wp)))
            if nbytes == 0:
                raise McError(MC_EINVAL, "invalid world parameters")
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            h = C.c_void_p()
            rc = L.mc_create(C.byref(wp), self.workspace.data_ptr(), nbytes,
                             C.c_void_p(self.stream.cuda_stream), C.byref(h))
            if rc != MC_OK:
                raise McError(rc, L.mc_last_error(None).decode())
            self.h = h
            self.N = 0
            if "offsets" in world:
                self.load_filaments(world)

    # -- mc_load_filaments: host numpy arrays or device tensors --
    def load_filaments(self, world: dict):
        torch = self.torch
        off = np.ascontiguousarray(world["offsets"], dtype=np.int32)
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            dev = []
            for k in _CHAIN_KEYS:
                a = world[k]
                if not isinstance(a, torch.Tensor):
                    a = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
                dev.append(a.to(self.device, dtype=torch.float32, non_blocking=False).contiguous())
            rc = load_library().mc_load_filaments(
                self.h, len(off) - 1, off.ctypes.data_as(C.POINTER(C.c_int32)),
                *[C.c_void_p(t.data_ptr()) for t in dev])
        self._check(rc)
        self.N = int(off[-1])
        if world.get("act_L_amp") is not None:
            self.set_length_actuation(world["act_L_amp"])

    def set_length_actuation(self, act_L_amp):
        """mc_set_length_actuation: [N] host numpy array or device tensor (None switches it off)."""
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            if act_L_amp is None:
                rc = load_library().mc_set_length_actuation(self.h, None)
            else:
                a = act_L_amp
                if not isinstance(a, torch.Tensor):
                    a = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
                d = a.to(self.device, dtype=torch.float32).contiguous()
                assert d.numel() == self.N
                rc = load_library().mc_set_length_actuation(self.h, C.c_void_p(d.data_ptr()))
        self._check(rc)

    def load_fluid(self, step: int, fdev=None):
        """mc_load_fluid: step counter and (optionally) the populations [9, ny, nx] as mc_read_state returns them."""
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            d = None
            if fdev is not None:
                if not isinstance(fdev, torch.Tensor):
                    fdev = torch.from_numpy(np.ascontiguousarray(fdev, dtype=np.float32))
                d = fdev.to(self.device, dtype=torch.float32).contiguous()
                assert d.numel() == 9 * self.nx * self.ny
            rc = load_library().mc_load_fluid(self.h, int(step), C.c_void_p(d.data_ptr()) if d is not None else None)
        self._check(rc)

    def set_positions(self, xy):
        """mc_set_positions: xy [N,2] host numpy array or device tensor, caller's bead order."""
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            if not isinstance(xy, torch.Tensor):
                xy = torch.from_numpy(np.ascontiguousarray(xy, dtype=np.float32))
            d = xy.to(self.device, dtype=torch.float32, non_blocking=False).contiguous()
            assert d.numel() == 2 * self.N
            rc = load_library().mc_set_positions(self.h, C.c_void_p(d.data_ptr()))
        self._check(rc)

    def step(self, n: int = 1):
        self._check(load_library().mc_step(self.h, int(n)))

    def read_state(self, keys=("xy", "u", "rho", "fdev", "field", "force", "sense"), host: bool = True):
        torch = self.torch
        ny, nx, N = self.ny, self.nx, self.N
        shapes = dict(xy=(N, 2), u=(2, ny, nx), rho=(ny, nx), fdev=(9, ny, nx),
                      field=(self.n_fields, ny, nx), force=(N, 2), sense=(N,))
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            out = {k: torch.empty(shapes[k], dtype=torch.float32, device=self.device) for k in keys}
            ptr = [C.c_void_p(out[k].data_ptr()) if k in out and out[k].numel() else None
                   for k in ("xy", "u", "rho", "fdev", "field", "force", "sense")]
            st = C.c_int64()
            rc = load_library().mc_read_state(self.h, C.byref(st), *ptr)
        self._check(rc)
        res = {k: (v.cpu().numpy() if host else v) for k, v in out.items()}
        res["step"] = int(st.value)
        return res

    def read_intermediates(self, host: bool = True):
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            rho_b = torch.empty((self.ny, self.nx), dtype=torch.float32, device=self.device)
            G = torch.empty((2, self.ny, self.nx), dtype=torch.float32, device=self.device)
            rc = load_library().mc_read_intermediates(self.h, C.c_void_p(rho_b.data_ptr()),
                                                      C.c_void_p(G.data_ptr()))
        self._check(rc)
        return dict(rho_b=rho_b.cpu().numpy() if host else rho_b, G=G.cpu().numpy() if host else G)

    def keep_intermediates(self, on: bool = True):
        self._check(load_library().mc_keep_intermediates(self.h, int(bool(on))))

    def texture_gathers(self, on: bool = True) -> bool:
        """mc_texture_gathers: returns whether the texture path is in use afterwards."""
        rc = load_library().mc_texture_gathers(self.h, int(bool(on)))
        if rc < 0:
            self._check(rc)
        return rc == 1

    def cluster_tiles(self, c: int = -1, all_tiles: bool = False) -> int:
        """mc_cluster_tiles: CTAs per crowded tile of the P2G kernels (0, 2, 4, 8; -1 automatic) -> in use.
        all_tiles: every tile gets a cluster in one launch (MC_CLUSTER_ALL_TILES) instead of the split launch."""
        rc = load_library().mc_cluster_tiles(self.h, int(c) | (64 if all_tiles and c >= 0 else 0))
        if rc < 0:
            self._check(rc)
        return rc

    def profile_enable(self, on: bool = True):
        self._check(load_library().mc_profile_enable(self.h, int(bool(on))))

    def profile_read(self):
        """-> ({slot name: summed ms}, number of captured steps)"""
        ms = (C.c_float * len(PROF_SLOTS))()
        n = C.c_int32()
        self._check(load_library().mc_profile_read(self.h, ms, C.byref(n)))
        return {k: float(ms[i]) for i, k in enumerate(PROF_SLOTS)}, int(n.value)

    def launch_count(self) -> int:
        return int(load_library().mc_launch_count(self.h))

    def _check(self, rc: int):
        if rc != MC_OK:
            raise McError(rc, load_library().mc_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            if self.owned:
                self.torch.cuda.synchronize(self.device)
                load_library().mc_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def deposit_noalloc(nx: int, ny: int, xy, out, stream=None):
    """mc_deposit_noalloc: rho_b = sum_i delta_h(g - X_i) into `out` (device float tensor [ny, nx]) from `xy`
    (device float tensor [N, 2]); the library's static scratch, no allocation.  Marshalling only: both
    tensors are the caller's.  Asynchronous on `stream` (a torch stream; default: the current one)."""
    import torch
    assert xy.is_cuda and out.is_cuda and xy.dtype == torch.float32 and out.dtype == torch.float32
    assert xy.is_contiguous() and out.is_contiguous() and out.numel() == nx * ny
    st = stream if stream is not None else torch.cuda.current_stream(xy.device)
    with torch.cuda.device(xy.device):
        rc = load_library().mc_deposit_noalloc(int(nx), int(ny), int(xy.shape[0]),
                                               C.c_void_p(xy.data_ptr()) if xy.numel() else None,
                                               C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream))
    if rc != MC_OK:
        raise McError(rc, load_library().mc_noalloc_last_error().decode())
    return out


class Batch:
    """mc_create_batch + mc_load_filaments_batch from a list of worlds.py dicts that share their
    parameters and chain structure (offsets); mc_step_batch; world(k) -> a World view for read-outs."""

    def __init__(self, worlds: list, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2607_02954_b200 needs a CUDA device (no CPU fallback)")
        L = load_library()
        self.torch = torch
        self.device = torch.device(device)
        self.p = worlds[0]["params"]
        self.n = len(worlds)
        self.h = None
        off = np.ascontiguousarray(worlds[0]["offsets"], dtype=np.int32)
        for w in worlds[1:]:
            if not np.array_equal(np.asarray(w["offsets"]), off):
                raise ValueError("the worlds of a batch must share their chain structure (offsets)")
        self.N = int(off[-1])
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            wp, keep = make_params(self.p)
            nbytes = int(L.mc_batch_workspace_bytes(C.byref(wp), self.n))
            if nbytes == 0:
                raise McError(MC_EINVAL, "invalid world parameters or batch size")
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            h = C.c_void_p()
            rc = L.mc_create_batch(C.byref(wp), self.n, self.workspace.data_ptr(), nbytes,
                                   C.c_void_p(self.stream.cuda_stream), C.byref(h))
            if rc != MC_OK:
                raise McError(rc, L.mc_batch_last_error(None).decode())
            self.h = h
            with torch.cuda.stream(self.stream):
                dev = []
                for k in _CHAIN_KEYS:
                    a = np.stack([np.ascontiguousarray(w[k], dtype=np.float32) for w in worlds])
                    dev.append(torch.from_numpy(a).to(self.device).contiguous())
                la = None
                if any(w.get("act_L_amp") is not None for w in worlds):
                    la = torch.from_numpy(np.stack([
                        np.ascontiguousarray(w["act_L_amp"] if w.get("act_L_amp") is not None else np.zeros(self.N),
                                             dtype=np.float32) for w in worlds])).to(self.device).contiguous()
                rc = L.mc_load_filaments_batch(
                    self.h, len(off) - 1, off.ctypes.data_as(C.POINTER(C.c_int32)),
                    *[C.c_void_p(t.data_ptr()) for t in dev], C.c_void_p(la.data_ptr()) if la is not None else None)
            self._check(rc)
        self._worlds = worlds

    def step(self, n: int = 1):
        self._check(load_library().mc_step_batch(self.h, int(n)))

    def set_positions(self, xy):
        """mc_set_positions_batch: xy [n, N, 2] host numpy array or device tensor."""
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            if not isinstance(xy, torch.Tensor):
                xy = torch.from_numpy(np.ascontiguousarray(xy, dtype=np.float32))
            d = xy.to(self.device, dtype=torch.float32, non_blocking=False).contiguous()
            assert d.numel() == 2 * self.N * self.n
            rc = load_library().mc_set_positions_batch(self.h, C.c_void_p(d.data_ptr()))
        self._check(rc)

    def read_positions(self, host: bool = True):
        """mc_read_positions_batch -> (xy [n, N, 2], step)"""
        torch = self.torch
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            out = torch.empty((self.n, self.N, 2), dtype=torch.float32, device=self.device)
            st = C.c_int64()
            rc = load_library().mc_read_positions_batch(self.h, C.byref(st), C.c_void_p(out.data_ptr()))
        self._check(rc)
        return (out.cpu().numpy() if host else out), int(st.value)

    def profile_enable(self, on: bool = True):
        """per-kernel CUDA-event timing of the batched launches (they are issued by world 0)"""
        L = load_library()
        self._check(L.mc_profile_enable(L.mc_batch_world(self.h, 0), int(bool(on))))

    def profile_read(self):
        L = load_library()
        ms = (C.c_float * len(PROF_SLOTS))()
        n = C.c_int32()
        self._check(L.mc_profile_read(L.mc_batch_world(self.h, 0), ms, C.byref(n)))
        return {k: float(ms[i]) for i, k in enumerate(PROF_SLOTS)}, int(n.value)

    def launch_count(self) -> int:
        L = load_library()
        return int(L.mc_launch_count(L.mc_batch_world(self.h, 0)))

    def world(self, k: int) -> "World":
        h = load_library().mc_batch_world(self.h, int(k))
        if not h:
            raise IndexError(k)
        return World(self._worlds[k], device=str(self.device), _member=(C.c_void_p(h), self.stream, self.N))

    def _check(self, rc: int):
        if rc != MC_OK:
            raise McError(rc, load_library().mc_batch_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            load_library().mc_destroy_batch(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

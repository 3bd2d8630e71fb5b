"""Batched small worlds: mc_create_batch /
mc_load_filaments_batch / mc_step_batch.  Every world of a batch must be BIT-EQUAL to the same
world stepped alone through mc_step; one world of every batch is also compared with the oracle."""
import numpy as np
import pytest

from paper_2607_02954_b200 import worlds
from test_gpu_parity import _varied, assert_close, rel_l2

pytestmark = pytest.mark.gpu

KEYS = ("xy", "u", "rho", "fdev", "force", "sense")


def family(make, n, **params):
    """n worlds of one recipe and chain structure, different seeds."""
    ws = [make(seed) for seed in range(n)]
    for w in ws:
        w["params"] = dict(w["params"], **params)
    return ws


def check_batch_equals_singles(ws, steps=(5, 7), keys=KEYS, oracle_world=1):
    from oracle import mco
    from paper_2607_02954_b200 import binding
    B = binding.Batch(ws)
    for s in steps:
        B.step(s)
    total = sum(steps)
    for k, w in enumerate(ws):
        S = binding.World(w)
        S.step(total)
        a, b = B.world(k).read_state(keys=keys), S.read_state(keys=keys)
        assert a["step"] == b["step"] == total
        for key in keys:
            assert a[key].tobytes() == b[key].tobytes(), (k, key)
        S.close()
    # and the batch agrees with the oracle (one world, trajectory bar)
    O = mco.World(ws[oracle_world])
    O.step(total)
    assert_close("batch world vs oracle", B.world(oracle_world).read_state(keys=("xy",))["xy"], O.read_state()["xy"], 1e-3)
    B.close()


def test_batch_of_uniform_worlds_is_bit_equal():
    # config-2 recipe at a quarter of the size: 64-bead chains, aligned windows, one-CTA K0
    ws = family(lambda s: worlds.random_world(128, 128, 64, 64, seed=s), 6)
    check_batch_equals_singles(ws)


def test_batch_of_ragged_worlds_with_both_fields_is_bit_equal():
    lengths = [3, 5, 16, 31, 33, 64, 65, 100]
    ws = family(lambda s: worlds.ragged_world(96, 64, lengths, seed=s, static_source=True), 5)
    # one world with per-bead parameters: the whole batch takes the general parameter path
    ws[2] = _varied(ws[2], 77)
    check_batch_equals_singles(ws)


def test_batch_with_one_crowded_world_is_bit_equal():
    # a crowded member widens the deposit CTAs (and would switch on tile clusters) for the whole batch
    ws = family(lambda s: worlds.random_world(64, 64, 96, 16, seed=s, kappa=0.25, kappa_rep=2e-4,
                                              clustered=3.0 if s == 1 else 0.0), 4)
    check_batch_equals_singles(ws, steps=(4, 4))


def test_batch_config1_worlds_is_bit_equal():
    # BASELINE.json config 1 (one 32-bead filament, 64 x 64): 16 individuals, different phases
    def make(seed):
        w = worlds.make_world("1")
        w["act_phase"] = (w["act_phase"] + np.float32(0.37 * seed)).astype(np.float32)
        w["xy"] = (w["xy"] + np.float32(1.7 * seed)).astype(np.float32)
        return w
    check_batch_equals_singles(family(make, 16), steps=(8, 9))


def test_batch_mdf_pbd_and_two_layer_variants_are_bit_equal():
    mk = lambda s: worlds.ragged_world(96, 64, [5, 16, 32, 33, 64, 90], seed=s)
    check_batch_equals_singles(family(mk, 3, coupling=1, mdf_iters=3), steps=(3, 4))
    check_batch_equals_singles(family(mk, 3, pbd_iters=3, pbd_order=1, pbd_project=1), steps=(3, 4))
    check_batch_equals_singles(family(mk, 3, two_layer=1), steps=(3, 4))


def test_batch_medium_worlds_cluster_k0_is_bit_equal():
    # 40,960 beads per world: the one-cluster K0 path, batched over blockIdx.y
    ws = family(lambda s: worlds.random_world(384, 384, 640, 64, seed=s), 3)
    check_batch_equals_singles(ws, steps=(4, 5), keys=("xy", "u", "force"))


def test_batch_members_cannot_be_stepped_alone_and_loads_are_checked():
    from paper_2607_02954_b200 import binding
    ws = family(lambda s: worlds.random_world(64, 64, 8, 16, seed=s), 3)
    B = binding.Batch(ws)
    lib = binding.load_library()
    h1 = lib.mc_batch_world(B.h, 1)
    assert lib.mc_step(h1, 1) == binding.MC_ESTATE
    assert lib.mc_batch_world(B.h, 3) is None and lib.mc_batch_world(B.h, -1) is None
    B.step(2)
    assert B.world(2).read_state(keys=("xy",))["step"] == 2
    B.close()
    bad = [dict(w) for w in ws]
    bad[1]["k_bend"] = bad[1]["k_bend"] * 3
    with pytest.raises(binding.McError) as e:
        binding.Batch(bad)
    assert e.value.code == binding.MC_EINVAL and "world 1" in str(e.value)
    # a load that fails part-way leaves the batch unusable until a good one
    import ctypes as C
    import torch
    B2 = binding.Batch(ws)
    dev = []
    for k in binding._CHAIN_KEYS:
        a = np.stack([np.ascontiguousarray(w[k], dtype=np.float32) for w in bad])
        dev.append(torch.from_numpy(a).cuda())
    off = np.ascontiguousarray(ws[0]["offsets"], dtype=np.int32)
    rc = lib.mc_load_filaments_batch(B2.h, len(off) - 1, off.ctypes.data_as(C.POINTER(C.c_int32)),
                                     *[C.c_void_p(t.data_ptr()) for t in dev], None)
    assert rc == binding.MC_EINVAL
    assert lib.mc_step_batch(B2.h, 1) == binding.MC_ESTATE
    B2.close()
    other = worlds.random_world(64, 64, 4, 32, seed=9)          # different chain structure
    with pytest.raises(ValueError):
        binding.Batch([ws[0], other])


def test_batch_set_positions_on_a_member():
    # a member's positions may be replaced between batch steps (per-world state only)
    from paper_2607_02954_b200 import binding
    ws = family(lambda s: worlds.random_world(96, 64, 12, 32, seed=s), 3)
    B = binding.Batch(ws)
    B.step(3)
    shifted = (B.world(1).read_state(keys=("xy",))["xy"] + np.float32(0.4)).astype(np.float32)
    B.world(1).set_positions(shifted)
    B.step(3)
    S = binding.World(ws[1])
    S.step(3)
    S.set_positions(shifted)
    S.step(3)
    a, b = B.world(1).read_state(keys=("xy", "u")), S.read_state(keys=("xy", "u"))
    assert a["xy"].tobytes() == b["xy"].tobytes() and a["u"].tobytes() == b["u"].tobytes()
    # the neighbours were not disturbed
    S0 = binding.World(ws[0])
    S0.step(6)
    assert B.world(0).read_state(keys=("xy",))["xy"].tobytes() == S0.read_state(keys=("xy",))["xy"].tobytes()


def test_batch_positions_in_one_call_each_way():
    # mc_set_positions_batch / mc_read_positions_batch = the per-world calls, bit for bit
    from paper_2607_02954_b200 import binding
    ws = family(lambda s: worlds.ragged_world(96, 64, [5, 16, 33, 64], seed=s), 4)
    B = binding.Batch(ws)
    B.step(3)
    xy, step = B.read_positions()
    assert step == 3 and xy.shape == (4, B.N, 2)
    for k in range(4):
        assert xy[k].tobytes() == B.world(k).read_state(keys=("xy",))["xy"].tobytes()
    new = (xy + np.float32(0.3) * np.arange(1, 5, dtype=np.float32)[:, None, None]).astype(np.float32)
    B.set_positions(new)
    B.step(4)
    got, _ = B.read_positions()
    for k in range(4):
        S = binding.World(ws[k])
        S.step(3)
        S.set_positions(new[k])
        S.step(4)
        assert got[k].tobytes() == S.read_state(keys=("xy",))["xy"].tobytes(), k
        S.close()
    B.close()

"""Row f4, second half: slab decomposition of ONE propagation along q_1 (paper_2509_25840_b200/sharding.py), world size 2
on gloo (CPU).  The engine here is built on the CPU oracle's right-hand side (tests may use it): each rank steps its slab
with a halo exchange before every RK stage; the owned planes must equal the single-rank propagation of the whole grid,
and the summed partial expectations the global one.  On GPUs the same SlabPropagator drives a CHFPE handle
(tests/test_gpu_parity.py::test_slab_*)."""
import os
import socket

import numpy as np
import pytest

import chfpe_inputs as ci
import oracle
from conftest import make_obs

torch = pytest.importorskip("torch")

CFG = ci.config("cfg3s", nq=[9, 6], np=[6, 7], depth=2)
NSTEPS, DT = 3, 5e-3


class OracleSlabEngine:
    """stage_input / rk4_stage / expect on numpy arrays in the canonical layout (q_1 is the slowest axis of an element,
    so q_1 planes are contiguous there too), Horner form of RK4 as in the CUDA path (reading R13)."""

    def __init__(self, cfg):
        self.o = oracle.RefCHFPE(cfg)
        self.shape = (self.o.K,) + self.o.shape
        self.y = np.zeros(self.shape)
        self.va = np.zeros(self.shape)
        self.vb = np.zeros(self.shape)

    def _arr(self, stage):
        return (self.y, self.va, self.vb, self.va)[stage]

    def stage_input(self, stage):
        a = self._arr(stage)
        return torch.from_numpy(a).view(a.shape[0], a.shape[1], -1)

    def rk4_stage(self, stage, dt):
        c = (dt / 4.0, dt / 3.0, dt / 2.0, dt)[stage]
        out = (self.va, self.vb, self.va, self.y)[stage]
        out[...] = self.y + c * self.o.rhs(self._arr(stage))

    def expect(self, obs):
        self.o.import_state(self.y)
        return [self.o.expect(obs)]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2509_25840_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        oracle.set_threads(1)
        loc, geo = sharding.slab_config(CFG, rank, world)
        eng = OracleSlabEngine(loc)
        prop = sharding.SlabPropagator(eng, geo, sharding.DistExchange())
        full = oracle.RefCHFPE(CFG)
        X = ci.seeded_state(CFG, [sum(n) for n in full.elements()], seed=21)
        eng.y[...] = prop.local_slice(X)
        prop.step(NSTEPS, DT)
        np.save(os.path.join(out, "own%d.npy" % rank), prop.owned(eng.y))
        al = make_obs(oracle, ci.observable("alpha", 2))
        np.save(os.path.join(out, "exp%d.npy" % rank), np.array([prop.expect_sum(al)]))
    finally:
        dist.destroy_process_group()


def test_slab_geometry():
    from paper_2509_25840_b200 import sharding
    for n in (5, 9, 16, 20):
        for world in (1, 2, 3):
            if n // world < sharding.HALO:
                continue
            got = []
            for r in range(world):
                lo, hi = sharding.slab_range(n, r, world)
                got += list(range(lo, hi))
            assert got == list(range(n))
    loc, (lo, hi, hl, hh) = sharding.slab_config(CFG, 1, 2)
    assert (lo, hi, hl, hh) == (5, 9, 2, 0) and loc["nq"][0] == 6
    h = (CFG["qmax"][0] - CFG["qmin"][0]) / 8
    assert abs(loc["qmin"][0] - (CFG["qmin"][0] + 3 * h)) < 1e-14 and abs(loc["qmax"][0] - CFG["qmax"][0]) < 1e-14
    with pytest.raises(ValueError):
        sharding.slab_config(ci.config("cfg3s", nq=[5, 6]), 0, 3)


def test_slab_propagation_world2_equals_single_rank(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    full = OracleSlabEngine(CFG)
    X = ci.seeded_state(CFG, [sum(n) for n in full.o.elements()], seed=21)
    full.y[...] = X
    for _ in range(NSTEPS):
        for st in range(4):
            full.rk4_stage(st, DT)
    got = np.concatenate([np.load(os.path.join(str(tmp_path), "own%d.npy" % r)) for r in range(2)], axis=1)
    assert got.shape == full.y.shape
    assert np.linalg.norm((got - full.y).ravel()) <= 1e-13 * np.linalg.norm(full.y.ravel())
    # the oracle's own classical RK4 gives the same step (Horner form = textbook form for a linear generator)
    o = oracle.RefCHFPE(CFG)
    o.import_state(X)
    o.step(NSTEPS, DT)
    assert np.linalg.norm((got - o.export_state()).ravel()) <= 1e-12 * np.linalg.norm(full.y.ravel())
    al = make_obs(oracle, ci.observable("alpha", 2))
    want = o.expect(al)
    for r in range(2):
        assert abs(np.load(os.path.join(str(tmp_path), "exp%d.npy" % r))[0] - want) <= 1e-12 * abs(want)

"""world_size-2 CPU test (gloo) of the t1-sharded 2D response: the gathered matrix equals the single-rank one.
The engine here is the CPU oracle (tests may use it); on GPUs the same helper drives paper_2509_25840_b200.CHFPE."""
import os
import socket

import numpy as np
import pytest

import chfpe_inputs as ci
import oracle
from conftest import make_obs

torch = pytest.importorskip("torch")

CFG = ci.config("cfg3s", nq=[7, 6], np=[6, 7], depth=2)
T1 = [0, 1, 3, 4, 6]
T2 = [0, 2, 3]
T3 = [1, 2]


def _obs():
    return [make_obs(oracle, ci.observable(k, 2)) for k in ("mu", "alpha", "alpha")]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2509_25840_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        oracle.set_threads(1)
        o = oracle.RefCHFPE(CFG)
        o.equilibrate()
        A, B, C = _obs()
        R = sharding.response_2d_sharded(o, A, B, C, T1, T2, 10 * CFG["dt"])
        np.save(os.path.join(out, "R%d.npy" % rank), R)
        o.equilibrate()
        R3 = sharding.response_3d_sharded(o, A, B, C, A, T1[:3], T2[:2], T3, 10 * CFG["dt"])
        np.save(os.path.join(out, "R3_%d.npy" % rank), R3)
    finally:
        dist.destroy_process_group()


def test_rows_for_rank_partition():
    from paper_2509_25840_b200 import sharding
    for n1 in (1, 5, 64):
        for world in (1, 2, 3, 8):
            got = sorted(i for r in range(world) for i in sharding.rows_for_rank(n1, r, world))
            assert got == list(range(n1))
    with pytest.raises(ValueError):
        sharding.rows_for_rank(4, 2, 2)


def test_response_2d_sharded_world2(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    o = oracle.RefCHFPE(CFG)
    o.equilibrate()
    A, B, C = _obs()
    full = o.response_2d(A, B, C, T1, T2, 10 * CFG["dt"])
    for r in range(2):
        R = np.load(tmp_path / ("R%d.npy" % r))
        assert R.shape == full.shape
        assert np.max(np.abs(R - full)) <= 1e-14 * np.max(np.abs(full))
    o.equilibrate()
    full3 = o.response_3d(A, B, C, A, T1[:3], T2[:2], T3, 10 * CFG["dt"])
    for r in range(2):
        R3 = np.load(tmp_path / ("R3_%d.npy" % r))
        assert R3.shape == full3.shape == (3, 2, 2)
        assert np.max(np.abs(R3 - full3)) <= 1e-14 * np.max(np.abs(full3))


HCFG = ci.config("cfg3s", nq=[9, 8], np=[3, 3], depth=2)


def _hermite_worker(rank, world, port, out):
    """Row f1: the same helper with a Hermite-representation engine (here its numpy oracle; on GPUs
    paper_2509_25840_b200.Hermite, whose response_2d has the same signature)."""
    import torch.distributed as dist
    from oracle import hermite
    from paper_2509_25840_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        o = hermite.RefHermite(HCFG)
        o.equilibrate()
        mu, al = ci.observable("mu", 2), ci.observable("alpha", 2)
        R = sharding.response_2d_sharded(o, mu, al, al, T1, T2, 10 * HCFG["dt"])
        np.save(os.path.join(out, "H%d.npy" % rank), R)
    finally:
        dist.destroy_process_group()


def test_hermite_response_2d_sharded_world2(tmp_path):
    import torch.multiprocessing as mp
    from oracle import hermite
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_hermite_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    o = hermite.RefHermite(HCFG)
    o.equilibrate()
    mu, al = ci.observable("mu", 2), ci.observable("alpha", 2)
    full = o.response_2d(mu, al, al, T1, T2, 10 * HCFG["dt"])
    assert np.max(np.abs(full)) > 0
    for r in range(2):
        R = np.load(tmp_path / ("H%d.npy" % r))
        assert R.shape == full.shape
        assert np.max(np.abs(R - full)) <= 1e-14 * np.max(np.abs(full))

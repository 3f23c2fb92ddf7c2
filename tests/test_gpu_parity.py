"""Parity of the CUDA path (through the C-ABI binding) with the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): per-step relative L2 <= 1e-12; response functions relative max
error <= 1e-8.  Operator-level checks use 1e-13.  All tests need a GPU (`-m gpu`).
"""
import os

import numpy as np
import pytest

import chfpe_inputs as ci
import oracle
from conftest import make_obs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def gpu_mod():
    import paper_2509_25840_b200 as P
    return P


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def both(cfg, batch=1):
    P = gpu_mod()
    return P.CHFPE(cfg, batch=batch), oracle.RefCHFPE(cfg)


def obs_pair(kind, M):
    d = ci.observable(kind, M)
    return make_obs(gpu_mod(), d), make_obs(oracle, d)


SMALL = [
    ("m1_sqrt", ci.config("cfg2", nq=[37], np=[41], depth=5)),
    ("m1_w_c2", ci.config("cfg2", nq=[33], np=[29], depth=3, gauge="w", scheme="central2")),
    ("m2_sqrt", ci.config("cfg3s", nq=[13, 11], np=[12, 14], depth=3)),
    ("m2_w", ci.config("cfg3s", nq=[9, 10], np=[11, 8], depth=2, gauge="w", mass=[1.0, 1.3])),
    ("m3_sqrt", ci.config("cfg4s8", nq=[7, 8, 6], np=[8, 6, 9], depth=3)),
    ("m3_w_c2", ci.config("cfg4s8", nq=[6, 5, 7], np=[5, 7, 6], depth=2, gauge="w", scheme="central2",
                          mass=[1.0, 0.8, 1.2])),
    ("m2_16_brick", ci.config("cfg3s", nq=[7, 9])),
    ("m2_48_brick_w", ci.config("cfg3", nq=[6, 5], depth=2, gauge="w", mass=[1.0, 1.3])),
    ("m3_cube8", ci.config("cfg4s8")),
    ("m3_cube12", ci.config("cfg4s12", nq=[5, 6, 7])),
    ("m3_cube16_w", ci.config("cfg4", nq=[5, 5, 6], gauge="w")),
    ("m3_cube20_c2", ci.config("cfg5", nq=[5, 5, 5], depth=2, scheme="central2")),
]


@pytest.mark.parametrize("name,cfg", SMALL, ids=[c[0] for c in SMALL])
def test_operator_step_kick_expect(name, cfg):
    g, o = both(cfg)
    M = cfg["n_modes"]
    assert g.elements() == o.elements() and g.K == o.K
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=1)
    g.import_state(X); o.import_state(X)
    assert np.array_equal(g.export_state(), X)                         # canonical round trip is exact
    # right-hand side of Eq. (8)
    Fg, Fo = g.export_rhs(), o.rhs(X)
    assert rel_l2(Fg, Fo) < 1e-13
    for k in range(o.K):
        assert np.linalg.norm(Fg[k] - Fo[k]) <= 1e-13 * np.linalg.norm(Fo)
    # expectation of a general observable (element 0 and a higher element)
    gen = dict(c0=0.3, lin_q=[0.7, -0.4, 0.2][:M], quad=[[0.5, 0.2, -0.1][:M], [0.1, -0.3, 0.25][:M], [0.05, 0.15, 0.4][:M]][:M],
               lin_p=[0.3, -0.2, 0.1][:M])
    og, oo = make_obs(gpu_mod(), gen), make_obs(oracle, gen)
    eg, eo = g.expect(og)[0], o.expect(oo)
    assert abs(eg - eo) <= 1e-12 * max(1.0, abs(eo))
    assert abs(g.expect_element(og, o.K - 1) - o.expect(oo, element=o.K - 1)) <= 1e-12 * max(1.0, abs(eo))
    # one step and ten steps
    g.step(1, cfg["dt"]); o.step(1, cfg["dt"])
    assert rel_l2(g.export_state(), o.export_state()) < 1e-12
    g.step(9, cfg["dt"]); o.step(9, cfg["dt"])
    assert rel_l2(g.export_state(), o.export_state()) < 1e-12
    # kick (Eq. 18) with a general observable
    g.import_state(X); o.import_state(X)
    g.kick(og); o.kick(oo)
    assert rel_l2(g.export_state(), o.export_state()) < 1e-13
    g.close()


@pytest.mark.parametrize("name,cfg", SMALL[:5], ids=[c[0] for c in SMALL[:5]])
def test_equilibrate(name, cfg):
    g, o = both(cfg)
    rg = g.equilibrate(3, cfg["dt"])
    ro = o.equilibrate(3, cfg["dt"])
    assert rel_l2(g.export_state(), o.export_state()) < 1e-12
    assert abs(rg - ro) <= 1e-9 * ro
    one_g, one_o = obs_pair("one", cfg["n_modes"])
    assert abs(g.expect(one_g)[0] - o.expect(one_o)) < 1e-12
    g.close()


def test_response_1d_config1_full():
    """BASELINE config 1 at full size: 2000 steps, <q> every step; also against the closed form."""
    cfg = ci.config("cfg1")
    g, o = both(cfg)
    mu_g, mu_o = obs_pair("mu", 1)
    g.equilibrate(); o.equilibrate()
    Rg = g.response_1d(mu_g, mu_g, 2001, 1, cfg["dt"])
    Ro = o.response_1d(mu_o, mu_o, 2001, 1, cfg["dt"])
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    r = np.roots([1.0, 1.0, 1.5, 1.0])
    dp = 3 * r * r + 2 * r + 1.5
    t = np.arange(2001) * cfg["dt"]
    bo = np.real(sum((ri + 1.0) / di * np.exp(ri * t) for ri, di in zip(r, dp)))
    assert np.max(np.abs(-Rg - bo)) < 6e-5            # h^4 error of the sqrt(W_eq) gauge on 64 x 64 (pin P1)
    g.close()


def test_response_1d_config2_full():
    """BASELINE config 2 at full size: 10^4 steps of dt = 5e-4, mu = q + 0.1 q^2, sampled every 10 steps."""
    cfg = ci.config("cfg2")
    g, o = both(cfg)
    mu_g, mu_o = obs_pair("mu_nl", 1)
    g.equilibrate(); o.equilibrate()
    Rg = g.response_1d(mu_g, mu_g, 1001, 10, cfg["dt"])
    Ro = o.response_1d(mu_o, mu_o, 1001, 10, cfg["dt"])
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    g.close()


@pytest.mark.parametrize("name,cfg,steps", [("cfg3s", ci.config("cfg3s"), {"mu": 2000, "alpha": 2000}),
                                            ("cfg4s8", ci.config("cfg4s8"), {"mu": 2000, "alpha": 400})])
def test_response_1d_shrunken_multimode(name, cfg, steps):
    """SURVEY 8(d) parity protocol (ii) on the shrunken multi-mode configurations 3' (16^4, 15 elements) and 4'
    (8^6, 20 elements): 2000 RK4 steps of the kicked state, sampled every 10 steps, rel-max <= 1e-8 (the step count
    is what the oracle affords: 40-90 ms per step on the box's cores; alpha on 4' runs 400 steps)."""
    g, o = both(cfg)
    M = cfg["n_modes"]
    for kind, nsteps in steps.items():
        a_g, a_o = obs_pair(kind, M)
        g.equilibrate(); o.equilibrate()
        Rg = g.response_1d(a_g, a_g, nsteps // 10 + 1, 10, cfg["dt"])
        Ro = o.response_1d(a_o, a_o, nsteps // 10 + 1, 10, cfg["dt"])
        assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro)), kind
    g.close()


@pytest.mark.parametrize("batch", [1, 2, 4])
def test_response_2d_batched(batch):
    """R2 (Eq. 16) with t1 replicas propagated together; batched == unbatched == oracle."""
    cfg = ci.config("cfg4s8", nq=[6, 6, 6], np=[6, 6, 6])
    g, o = both(cfg, batch=batch)
    mu_g, mu_o = obs_pair("mu", 3)
    al_g, al_o = obs_pair("alpha", 3)
    t1 = [0, 2, 3, 7, 8, 12, 16, 20]; t2 = [0, 1, 4, 6, 9, 13, 18, 24, 30]      # 20 + 8 x 30 = 260 replica-steps
    g.equilibrate(); o.equilibrate()
    Rg = g.response_2d(mu_g, al_g, al_g, t1, t2, cfg["dt"] * 10)
    Ro = o.response_2d(mu_o, al_o, al_o, t1, t2, cfg["dt"] * 10)
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    if batch > 1:
        g1 = gpu_mod().CHFPE(cfg, batch=1)
        g1.equilibrate()
        R1 = g1.response_2d(mu_g, al_g, al_g, t1, t2, cfg["dt"] * 10)
        assert np.max(np.abs(Rg - R1)) <= 1e-14 * np.max(np.abs(R1))
        g1.close()
    g.close()


def test_batched_step_equals_single():
    cfg = ci.config("cfg3s", nq=[10, 9], np=[9, 10], depth=2)
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=3)
    o = oracle.RefCHFPE(cfg)
    levels = [sum(n) for n in o.elements()]
    Xs = [ci.seeded_state(cfg, levels, seed=s) for s in range(3)]
    for b in range(3):
        g.import_state(Xs[b], replica=b)
    g.step(4, cfg["dt"])
    mu_g, mu_o = obs_pair("mu", 2)
    e = g.expect(mu_g)
    for b in range(3):
        o.import_state(Xs[b]); o.step(4, cfg["dt"])
        assert rel_l2(g.export_state(b), o.export_state()) < 1e-12
        assert abs(e[b] - o.expect(mu_o)) <= 1e-12 * max(1.0, abs(o.expect(mu_o)))
    g.close()


@pytest.mark.parametrize("coop", ["0", "2"])
def test_cooperative_and_per_stage_paths_agree(monkeypatch, coop):
    """Persistent cooperative multi-step kernel (CHFPE_COOP=2: every L2-resident state) vs per-stage launches
    (CHFPE_COOP=0): both against the oracle, M = 1, 2, 3."""
    monkeypatch.setenv("CHFPE_COOP", coop)
    for cfg in (ci.config("cfg2", nq=[37], np=[41], depth=5), ci.config("cfg3s", nq=[9, 10], np=[11, 8], depth=2),
                ci.config("cfg4s8", nq=[6, 5, 7], np=[8, 8, 8], depth=2)):
        g, o = both(cfg)
        M = cfg["n_modes"]
        mu_g, mu_o = obs_pair("mu_nl", M)
        g.equilibrate(); o.equilibrate()
        Rg = g.response_1d(mu_g, mu_g, 7, 3, cfg["dt"])
        Ro = o.response_1d(mu_o, mu_o, 7, 3, cfg["dt"])
        assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
        assert rel_l2(g.export_state(), o.export_state()) < 1e-12
        assert (g.launch_count() < 40) if coop == "2" else (g.launch_count() > 60)
        g.close()


FAMILY_ENVS = [
    ({}, "tma"),                                                       # default for three modes with CENTRAL4
    ({"CHFPE_TMA": "0"}, "brick"),                                     # the register-staged brick kernel of round 1
    ({"CHFPE_TMA_RING": "0", "CHFPE_TMA_SLOTS": "4"}, None),           # q_3 neighbours as chunks instead of the ring
    ({"CHFPE_TMA_NPART": "1"}, None),                                  # whole bricks per chunk (no halo-plane kind)
    ({"CHFPE_TMA_SLOTS": "4"}, None),                                  # four ring slots
]


@pytest.mark.parametrize("name", ["cfg4", "cfg5"])
def test_stage_kernel_is_bitwise_reproducible_at_full_size(name):
    """k_stage_tma synchronises its warps with mbarriers only (ring slots, exchange planes, the edge buffer of the p_3 stencil
    at 20^3): a missing wait would be a race, i.e. run-to-run differences, most likely with every CTA of the bench workload
    in flight.  No atomics, fixed summation order: the right-hand side of the same state must come out BITWISE equal twice,
    and so must two RK4 steps (the last stage updates y in place)."""
    cfg = ci.config(name)
    P = gpu_mod()
    arr = 8.0 * np.prod(cfg["nq"]) * np.prod(cfg["np"]) * 20           # one state array; the workspace holds three, the test three more
    if torch.cuda.mem_get_info()[0] < 6.5 * arr + 2e9:
        pytest.skip("needs %.0f GB of device memory" % ((6.5 * arr + 2e9) / 1e9))
    g = P.CHFPE(cfg)
    assert g.stage_kernel() == "tma"
    g.equilibrate(residual=False)
    g.kick(make_obs(P, ci.observable("mu", 3)))
    g.step(1, cfg["dt"])                       # a state that is non-trivial on every element
    X = g.export_state_device().clone()
    F1 = g.export_rhs_device().clone()
    F2 = g.export_rhs_device()
    assert torch.equal(F1, F2) and bool(torch.isfinite(F1).all()) and float(F1.abs().max()) > 0.0
    del F1, F2
    g.step(2, cfg["dt"])
    Y1 = g.export_state_device().clone()
    g.import_state(X)
    g.step(2, cfg["dt"])
    assert torch.equal(Y1, g.export_state_device())
    g.close()


@pytest.mark.parametrize("name", ["m2_48_brick_w", "m3_cube12", "m3_cube20_c2"])
def test_expectation_kernels_agree(name, monkeypatch):
    """k_expect_pbrick (momentum factors of the observable and of the gauge weight tabulated per brick in shared memory; the
    default for p-bricks of 256 ... 8192 cells) against the generic reduction (CHFPE_EXPECT_PBRICK=0) and the oracle, on
    element 0 and on the last element, both gauges, two batch slots, general observable incl. the momentum part."""
    cfg = dict(SMALL)[name]
    M = cfg["n_modes"]
    gen = dict(c0=-0.2, lin_q=[0.7, -0.4, 0.2][:M], quad=[[0.5, 0.2, -0.1][:M], [0.1, -0.3, 0.25][:M], [0.05, 0.15, 0.4][:M]][:M],
               lin_p=[0.3, -0.2, 0.1][:M])
    og, oo = make_obs(gpu_mod(), gen), make_obs(oracle, gen)
    g, o = both(cfg, batch=2)
    X = ci.seeded_state(cfg, [sum(n) for n in o.elements()], seed=6)
    g.import_state(X); g.import_state(-3.0 * X, replica=1); o.import_state(X)
    ref0, refK = o.expect(oo), o.expect(oo, element=o.K - 1)
    monkeypatch.setenv("CHFPE_EXPECT_PBRICK", "0")
    g0 = gpu_mod().CHFPE(cfg, batch=2)
    g0.import_state(X); g0.import_state(-3.0 * X, replica=1)
    for h in (g, g0):
        e = h.expect(og)
        assert abs(e[0] - ref0) <= 1e-12 * max(1.0, abs(ref0)) and abs(e[1] + 3.0 * ref0) <= 3e-12 * max(1.0, abs(ref0))
        assert abs(h.expect_element(og, o.K - 1) - refK) <= 1e-12 * max(1.0, abs(ref0))
    assert abs(g.expect(og)[0] - g0.expect(og)[0]) <= 1e-13 * max(1.0, abs(ref0))
    g.close(); g0.close()


@pytest.mark.parametrize("env,family", FAMILY_ENVS, ids=["-".join("%s%s" % (k[6:], v) for k, v in e.items()) or "default"
                                                         for e, _ in FAMILY_ENVS])
def test_stage_kernel_families(monkeypatch, env, family):
    """Every stage-kernel family and variant of the three-mode CENTRAL4 path computes the same right-hand side and steps:
    the bulk-copy fed kernel (k_stage_tma: ring / no ring along q_3, bricks cut in two parts or whole, 4 / 5 slots) and the
    brick kernel (k_stage_brick3), on all four instantiated brick shapes, with ragged q grids so that every edge case of
    the chunk stream occurs (ghost bricks on all axes, lines shorter than the ring depth + 2)."""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    for cfg in (ci.config("cfg4s8", nq=[6, 5, 7]), ci.config("cfg4", nq=[5, 6, 5], depth=2),
                ci.config("cfg4s12", nq=[5, 5, 6], depth=2), ci.config("cfg5", nq=[5, 5, 6], depth=1),
                ci.config("cfg4", nq=[5, 5, 19], depth=1)):
        g, o = both(cfg, batch=2)
        if family is not None:
            assert g.stage_kernel() == family, (cfg["name"], g.stage_kernel())
        else:
            assert g.stage_kernel() in ("tma", "brick")                # (a variant without an instantiation: brick kernel)
        levels = [sum(n) for n in o.elements()]
        X = ci.seeded_state(cfg, levels, seed=4)
        g.import_state(X); g.import_state(X, replica=1); o.import_state(X)
        Fg, Fo = g.export_rhs(1), o.rhs(X)
        assert rel_l2(Fg, Fo) < 1e-13
        for k in range(o.K):
            assert np.linalg.norm(Fg[k] - Fo[k]) <= 1e-13 * np.linalg.norm(Fo)
        g.step(3, cfg["dt"]); o.step(3, cfg["dt"])
        assert rel_l2(g.export_state(0), o.export_state()) < 1e-12
        assert rel_l2(g.export_state(1), o.export_state()) < 1e-12
        g.close()


@pytest.mark.parametrize("name", ["cfg3", "cfg4", "cfg5"])
def test_full_size_sampled_rhs_and_step_properties(name):
    """BASELINE configs 3 and 4 at full size, in the launch configuration bench.py times: sampled entries of the
    right-hand side against the oracle's point formula, plus size-independent properties of a step."""
    cfg = ci.config(name)
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=1)
    assert g.stage_kernel() in ("brick", "tma")      # the named configurations must not fall back to the generic kernel
    o = oracle.RefCHFPE(cfg)
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=0)
    g.import_state(X)
    F = g.export_rhs()
    rng = np.random.default_rng(5)
    Ff = F.reshape(o.K, -1)
    scale = float(np.sqrt(np.mean(Ff[:, ::997] ** 2)))
    shape = o.shape
    samples = [(int(rng.integers(o.K)), int(rng.integers(o.cells))) for _ in range(3000)]
    # add corners / edges of the grid (zero-ghost boundary handling)
    for k in (0, o.K - 1):
        for cell in (0, o.cells - 1, shape[-1] - 1, o.cells - shape[-1], o.cells // 2):
            samples.append((k, cell))
    worst = 0.0
    for k, cell in samples:
        worst = max(worst, abs(Ff[k, cell] - o.rhs_at(X, k, cell)))
    assert worst <= 1e-12 * scale
    # properties of one full-size step: the scaled norm must not grow (sqrt gauge, pin P6) and <1> drifts by O(dt h^4)
    one_g, _ = obs_pair("one", cfg["n_modes"])
    n0 = g.expect(one_g)[0]
    g.step(2, cfg["dt"])
    Y = g.export_state()
    w = []
    for n in o.elements():
        f = 1.0
        for s, ns in enumerate(n):
            for j in range(1, ns + 1):
                f *= j * cfg["zeta"][s] * cfg["gamma"][s] * cfg["mass"][s] / cfg["beta"]
        w.append(f)
    norm = lambda Z: sum(float(np.sum(Z[k] ** 2)) / w[k] for k in range(o.K))
    assert norm(Y) <= norm(X) * (1 + 1e-12)
    assert np.all(np.isfinite(Y))
    assert abs(g.expect(one_g)[0] - n0) < 1e-2 * abs(n0)
    g.close()


def _per_element_rel_l2(A, B):
    """Overall rel-L2 and the worst element block, normalised by the block of the reference (SURVEY 8(d) protocol (i))."""
    K = B.shape[0]
    num = np.array([float(np.sum((A[k] - B[k]) ** 2)) for k in range(K)])
    den = np.array([float(np.sum(B[k] ** 2)) for k in range(K)])
    return float(np.sqrt(num.sum() / den.sum())), float(np.sqrt(np.max(num / den)))


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_full_size_one_step_parity(name):
    """SURVEY 8(d) parity protocol (i) at FULL size, in the launch configuration bench.py times: the whole right-hand
    side and one whole RK4 step of BASELINE configs 3 (48^4 x 15 elements, 8.0e7 values) and 4 (16^6 x 20 elements,
    3.4e8 values) against the oracle, element-wise: rel-L2 <= 1e-13 / 1e-12 overall AND for every element block."""
    cfg = ci.config(name)
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=1)
    assert g.stage_kernel() in ("brick", "tma")
    o = oracle.RefCHFPE(cfg)
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=2)
    g.import_state(X)
    F, Fo = g.export_rhs(), o.rhs(X)
    tot, blk = _per_element_rel_l2(F, Fo)
    assert tot < 1e-13 and blk < 1e-13, (tot, blk)
    del F, Fo
    o.import_state(X)
    del X
    g.step(1, cfg["dt"]); o.step(1, cfg["dt"])
    tot, blk = _per_element_rel_l2(g.export_state(), o.export_state())
    assert tot < 1e-12 and blk < 1e-12, (tot, blk)
    g.close()


def test_full_size_rhs_parity_config5():
    """BASELINE config 5 (20^6 x 20 elements = 1.28e9 values, 10.2 GB per array, one replica): the whole right-hand side
    against the oracle, per element block.  Needs about 60 GB of host memory (state, two right-hand sides, the oracle's
    copy) and 25 GB on the device; skipped, with the reason, where that is not available -- the sampled-entry test
    above then remains the full-size check of this configuration."""
    import psutil
    import torch
    cfg = ci.config("cfg5")
    if psutil.virtual_memory().available < 70e9:
        pytest.skip("full-array config-5 comparison not run: needs 70 GB of free host memory, %.0f GB available"
                    % (psutil.virtual_memory().available / 1e9))
    if torch.cuda.mem_get_info()[0] < 45e9:
        pytest.skip("full-array config-5 comparison not run: needs 45 GB of device memory")
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=1)
    o = oracle.RefCHFPE(cfg)
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=3)
    g.import_state(X)
    Fo = o.rhs(X)
    del X
    F = g.export_rhs()
    tot, blk = _per_element_rel_l2(F, Fo)
    print("config 5 full-array RHS ran: rel-L2 %.2e overall, %.2e worst element block" % (tot, blk))
    assert tot < 1e-13 and blk < 1e-13, (tot, blk)
    g.close()


def test_error_paths():
    P = gpu_mod()
    bad = ci.config("cfg1", nq=[3])
    with pytest.raises(P.ChfpeError):
        P.CHFPE(bad)
    with pytest.raises(P.ChfpeError):
        P.CHFPE(ci.config("cfg1", depth=-1))
    g = P.CHFPE(ci.config("cfg1"))
    mu_g, _ = obs_pair("mu", 1)
    with pytest.raises(P.ChfpeError):
        g.response_1d(mu_g, mu_g, 3, 1, 1e-3)          # before equilibrate / import
    g.equilibrate()
    with pytest.raises(P.ChfpeError):
        g.response_2d(mu_g, mu_g, mu_g, [3, 1], [0], 1e-3)   # unsorted t1
    g.close()


def test_degenerate_and_edge_cases():
    """Depth 0 (one element, no hierarchy links), minimum 5-point axes, zeta = 0, zero steps, zero stride,
    repeated delays, more replica slots than t1 rows, n_samples = 0."""
    mu1_g, mu1_o = obs_pair("mu", 1)
    # depth 0 on a 5 x 5 grid: pure Liouvillian, K = 1
    cfg = ci.config("cfg1", nq=[5], np=[5], depth=0)
    g, o = both(cfg)
    assert g.K == 1
    X = ci.seeded_state(cfg, [0], seed=2)
    g.import_state(X); o.import_state(X)
    assert rel_l2(g.export_rhs(), o.rhs(X)) < 1e-13
    g.step(0, cfg["dt"])                                       # no-op
    assert np.array_equal(g.export_state(), X)
    g.step(5, cfg["dt"]); o.step(5, cfg["dt"])
    assert rel_l2(g.export_state(), o.export_state()) < 1e-12
    assert g.response_1d(mu1_g, mu1_g, 0, 1, cfg["dt"]).size == 0
    g.close()
    # zeta = 0: the hierarchy decouples downwards (rigid rotation, pin P5), stride 0 repeats the same sample
    cfg = ci.config("cfg1", nq=[21], np=[23], depth=2, zeta=[0.0])
    g, o = both(cfg)
    g.equilibrate(); o.equilibrate()
    p_g, p_o = (m.make_observable(0.0, [0.0], [[0.0]], [1.0]) for m in (gpu_mod(), oracle))   # C = p: <p>(0+) = -1
    Rg = g.response_1d(mu1_g, p_g, 4, 0, cfg["dt"])
    Ro = o.response_1d(mu1_o, p_o, 4, 0, cfg["dt"])
    assert abs(Ro[0] + 1.0) < 5e-3                              # h^4 error of the 21 x 23 grid
    assert np.allclose(Rg, Rg[0], rtol=1e-13, atol=0) and np.max(np.abs(Rg - Ro)) <= 1e-12
    g.close()
    # 2D: repeated t1 / t2 entries, batch larger than the number of rows
    cfg = ci.config("cfg3s", nq=[6, 7], np=[7, 6], depth=2)
    g, o = both(cfg, batch=4)
    mu_g, mu_o = obs_pair("mu", 2)
    al_g, al_o = obs_pair("alpha", 2)
    g.equilibrate(); o.equilibrate()
    t1, t2 = [0, 0, 2], [0, 3, 3, 5]
    Rg = g.response_2d(mu_g, al_g, mu_g, t1, t2, 10 * cfg["dt"])
    Ro = o.response_2d(mu_o, al_o, mu_o, t1, t2, 10 * cfg["dt"])
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    assert np.array_equal(Rg[0], Rg[1]) and np.array_equal(Rg[:, 1], Rg[:, 2])
    g.close()


def test_two_dimensional_closed_form_on_gpu():
    """Pin P4 on the CUDA path itself: harmonic + LL, A = C = q, B = q^2 in the W gauge:
    R2_lib(t2, t1) = 2 R_phys(t1) R_phys(t2) (tests/golden/r2_closed_form.txt)."""
    cfg = ci.config("cfg1", nq=[48], np=[48], depth=4, gauge="w")
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=2)
    q = P.make_observable(0.0, [1.0], [[0.0]], [0.0])
    q2 = P.make_observable(0.0, [0.0], [[2.0]], [0.0])
    g.equilibrate()
    R = g.response_2d(q, q2, q, [800], [1200], 1e-3)
    assert abs(R[0, 0] - 1.153396427) < 2e-6
    g.close()


@pytest.mark.parametrize("name,batch", [("m1", 3), ("m2", 4), ("m3", 5)])
def test_response_3d(name, batch):
    """Row f2: R3 (Eq. 17) with the replicas of (batch-1)/2 t1 samples propagated together (ragged last group,
    repeated delays; batch-1 replicas when there is a single waiting time t2) against the oracle's plain triple loop;
    M = 1, 2, 3."""
    cfg = {"m1": ci.config("cfg2", nq=[37], np=[41], depth=4),
           "m2": ci.config("cfg3s", nq=[9, 10], np=[11, 8], depth=2),
           "m3": ci.config("cfg4s8", nq=[6, 5, 7], np=[5, 7, 6], depth=2)}[name]
    M = cfg["n_modes"]
    g, o = both(cfg, batch=batch)
    mu_g, mu_o = obs_pair("mu", M)
    al_g, al_o = obs_pair("alpha", M)
    nl_g, nl_o = obs_pair("mu_nl", M)
    g.equilibrate(); o.equilibrate()
    t1, t2, t3 = [0, 2, 5], [0, 1, 1, 4, 6], [0, 3, 4]
    dt = 10 * cfg["dt"]
    Rg = g.response_3d(mu_g, al_g, nl_g, al_g, t1, t2, t3, dt)
    Ro = o.response_3d(mu_o, al_o, nl_o, al_o, t1, t2, t3, dt)
    assert Rg.shape == (3, 5, 3)
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    assert np.array_equal(Rg[:, 1], Rg[:, 2])
    # replica 0 holds the t1 trajectory at its last delay; the call can be repeated after equilibrate
    g.equilibrate()
    Rg2 = g.response_3d(mu_g, al_g, nl_g, al_g, t1, t2, t3, dt)
    assert np.array_equal(Rg, Rg2)
    g.equilibrate()
    Rw = g.response_3d(mu_g, al_g, nl_g, al_g, t1, [4], t3, dt)      # fixed waiting time: C applied in place
    assert np.max(np.abs(Rw[:, 0] - Ro[:, 3])) <= 1e-8 * np.max(np.abs(Ro))
    g.close()


def test_response_3d_closed_forms_and_errors():
    """Pin P4b on the CUDA path: harmonic + LL in the W gauge, c = R_phys:
    A = D = q, B = C = q^2: -4 c(t1) c(t2) c(t3);  A = B = q, C = D = q^2: -4 c(t3)[c(t2) c(t1+t2+t3) + c(t2+t3) c(t1+t2)]."""
    cfg = ci.config("cfg1", nq=[48], np=[48], depth=4, gauge="w")
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=4)
    q = P.make_observable(0.0, [1.0], [[0.0]], [0.0])
    q2 = P.make_observable(0.0, [0.0], [[2.0]], [0.0])

    def c(t, w0=1.0, zeta=0.5, gamma=1.0):          # Brownian-oscillator response (3 x 3 first-moment ODE, pin P3)
        import scipy.linalg
        A = np.array([[0, 1, 0], [-w0 ** 2, 0, 1], [0, -zeta * gamma, -gamma]], dtype=float)
        return float(scipy.linalg.expm(t * A)[0, 1])

    t1, t2, t3 = [500], [300, 700], [400, 900]
    g.equilibrate()
    Ra = g.response_3d(q, q2, q2, q, t1, t2, t3, 1e-3)
    g.equilibrate()
    Rb = g.response_3d(q, q, q2, q2, t1, t2, t3, 1e-3)
    for j, b in enumerate(t2):
        for l, d in enumerate(t3):
            a_, b_, d_ = 0.5, b * 1e-3, d * 1e-3
            assert abs(Ra[0, j, l] + 4 * c(a_) * c(b_) * c(d_)) < 3e-5
            assert abs(Rb[0, j, l] + 4 * c(d_) * (c(b_) * c(a_ + b_ + d_) + c(b_ + d_) * c(a_ + b_))) < 3e-5
    with pytest.raises(Exception):
        g.response_3d(q, q2, q2, q, [3, 1], t2, t3, 1e-3)        # descending t1
    g.close()
    g2 = P.CHFPE(cfg, batch=2)
    g2.equilibrate()
    with pytest.raises(Exception):
        g2.response_3d(q, q2, q2, q, t1, t2, t3, 1e-3)           # two waiting times need three slots
    g2.equilibrate()
    Rw = g2.response_3d(q, q2, q2, q, t1, [700], t3, 1e-3)       # one waiting time runs in two
    assert np.max(np.abs(Rw[:, 0] - Ra[:, 1])) <= 1e-12
    g2.close()


PLAN_ENVS = [
    {"CHFPE_Q2CHUNK": "3", "CHFPE_GROUP": "3"},                      # ragged q_2 chunks (7 = 3 + 3 + 1 -> equalised), ragged last group
    {"CHFPE_Q2CHUNK": "2", "CHFPE_GROUP": "1", "CHFPE_BPC": "1"},
    {"CHFPE_BPC": "5"},                                              # n_q3 = 5: one run per q_3 line
    {"CHFPE_GROUP": "20"},                                           # all elements in one group
    {"CHFPE_L2MODE": "0"}, {"CHFPE_L2MODE": "3"},
    {"CHFPE_BRICK": "0"},                                            # generic kernel on a brick-shaped grid
]


@pytest.mark.parametrize("env", PLAN_ENVS, ids=["-".join("%s%s" % (k[6:], v) for k, v in e.items()) for e in PLAN_ENVS])
@pytest.mark.parametrize("shape", ["cube8", "cube20_two_pass", "m2_16"])
def test_brick_plan_variants(monkeypatch, env, shape):
    """The host-tabulated brick order (element groups, q_2 chunks, runs per CTA) and the L2 policies only change the
    ORDER and caching of the work: every variant must reproduce the oracle's right-hand side and steps.  (At full
    size configs 4 and 5 take the chunked / grouped paths that small grids would otherwise never reach.)"""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    cfg = {"cube8": ci.config("cfg4s8", nq=[6, 7, 5]),
           "cube20_two_pass": ci.config("cfg5", nq=[5, 6, 5], depth=2),
           "m2_16": ci.config("cfg3s", nq=[7, 10])}[shape]
    g, o = both(cfg, batch=2)
    if env.get("CHFPE_BRICK") == "0":
        assert g.stage_kernel() == "generic"
    else:
        assert g.stage_kernel() in ("brick", "tma")
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=11)
    g.import_state(X); g.import_state(X, replica=1); o.import_state(X)
    assert rel_l2(g.export_rhs(1), o.rhs(X)) < 1e-13
    g.step(2, cfg["dt"]); o.step(2, cfg["dt"])
    assert rel_l2(g.export_state(0), o.export_state()) < 1e-12
    assert np.array_equal(g.export_state(0), g.export_state(1))
    g.close()


GUARDED = [
    ("m3_cube8", ci.config("cfg4s8"), 2),
    ("m3_cube16", ci.config("cfg4", nq=[5, 5, 6]), 3),
    ("m3_cube20_two_pass", ci.config("cfg5", nq=[5, 5, 5], depth=2), 3),
    ("m2_48", ci.config("cfg3", nq=[6, 5], depth=2), 3),
    ("m3_generic", ci.config("cfg4s8", nq=[7, 8, 6], np=[8, 6, 9], depth=3), 4),
    ("m1_coop", ci.config("cfg1"), 2),
    ("m3_compact_transposing", ci.config("cfg4s8", nq=[8, 5, 6], np=[5, 8, 12], depth=2, scheme="compact6"), 3),
    ("m2_compact", ci.config("cfg3s", nq=[9, 10], np=[11, 8], depth=2, scheme="compact6"), 3),
]


@pytest.mark.parametrize("name,cfg,batch", GUARDED, ids=[c[0] for c in GUARDED])
def test_no_write_outside_the_workspace(name, cfg, batch):
    """Canary bytes on both sides of the caller-owned workspace survive every entry point, for every kernel family
    (brick single- and two-pass, two-mode view, generic, cooperative, COMPACT6 line and transposing kernels)."""
    P = gpu_mod()
    M = cfg["n_modes"]
    g = P.CHFPE(cfg, batch=batch, guard_bytes=1 << 20)
    mu, al = make_obs(P, ci.observable("mu", M)), make_obs(P, ci.observable("alpha", M))
    g.equilibrate(n_steps=2, dt=cfg["dt"])
    g.kick(mu); g.step(3, cfg["dt"]); g.expect(al)
    g.equilibrate()
    g.response_1d(mu, mu, 4, 2, cfg["dt"])
    g.equilibrate()
    g.response_2d(mu, al, al, [0, 1, 3], [0, 2], cfg["dt"])
    if batch >= 3:
        g.equilibrate()
        g.response_3d(mu, al, al, mu, [0, 2], [1, 2], [0, 1], cfg["dt"])
    X = g.export_state(batch - 1)
    g.import_state(X, replica=batch - 1)
    g.export_rhs()
    assert g.guards_intact()
    g.close()


COMPACT = [
    ("m1", ci.config("cfg2", nq=[37], np=[41], depth=4, scheme="compact6")),
    ("m2_w", ci.config("cfg3s", nq=[9, 10], np=[11, 8], depth=2, scheme="compact6", gauge="w")),
    ("m3", ci.config("cfg4s8", nq=[6, 5, 7], np=[5, 7, 6], depth=2, scheme="compact6")),
    # shapes whose contiguous p axis takes the transposing kernel (n <= 32, cells a multiple of 32 n)
    ("m1_t", ci.config("cfg2", nq=[32], np=[16], depth=3, scheme="compact6")),
    ("m2_t", ci.config("cfg3s", nq=[8, 7], np=[8, 16], depth=2, scheme="compact6")),
    ("m3_t", ci.config("cfg4s8", nq=[8, 5, 6], np=[5, 8, 12], depth=2, scheme="compact6", gauge="w")),
    # 24 and 32 points on the contiguous axis: the transposing kernel needs > 48 KB of dynamic shared memory
    ("m1_t32", ci.config("cfg2", nq=[32], np=[32], depth=3, scheme="compact6")),
    ("m2_t24", ci.config("cfg3s", nq=[8, 8], np=[8, 24], depth=2, scheme="compact6")),
    # 16^3 bricks (config 4's): the compile-time-shaped brick pass k_compact_pbrick<3, 8, 16>
    ("m3_cube16", ci.config("cfg4", nq=[5, 6, 5], depth=2, scheme="compact6", mass=[1.0, 0.8, 1.2])),
    # 48^2 (config 3) and 20^3 (config 5) bricks: k_compact_pbrick<2, 8, 48> (288 threads) and <3, 16, 20> (16 cells per thread)
    ("m2_sq48_w", ci.config("cfg3", nq=[6, 5], depth=2, scheme="compact6", gauge="w", mass=[1.0, 1.3])),
    ("m3_cube20", ci.config("cfg5", nq=[5, 5, 5], depth=1, scheme="compact6")),
    # 16 x 16 and 20 x 20 (q_2, q_3) planes: the fused plane pass k_compact_qplane (q_2 and q_3 in one launch)
    ("m3_qplane16_w", ci.config("cfg4s8", nq=[5, 16, 16], np=[5, 8, 8], depth=2, scheme="compact6", gauge="w", mass=[1.0, 0.8, 1.2])),
    ("m3_qplane20", ci.config("cfg4s8", nq=[6, 20, 20], np=[5, 8, 6], depth=1, scheme="compact6")),
    # 16- and 20-point q lines outside the plane pass: k_compact_qline (loads ahead of the recurrence), two and three modes
    ("m3_qline16", ci.config("cfg4s8", nq=[16, 5, 6], np=[5, 6, 7], depth=2, scheme="compact6", mass=[1.0, 0.8, 1.2])),
    ("m2_qline20_16_w", ci.config("cfg3s", nq=[20, 16], np=[9, 8], depth=2, scheme="compact6", gauge="w")),
    # 48-point q lines of two modes (config 3): k_compact_qline_long (window of three blocks of 8 points), both axes
    ("m2_qline48", ci.config("cfg3s", nq=[48, 48], np=[5, 6], depth=1, scheme="compact6", mass=[1.0, 1.3])),
]


@pytest.mark.parametrize("name,cfg", COMPACT, ids=[c[0] for c in COMPACT])
def test_compact6_path(name, cfg):
    """Step a9: Pade sixth-order derivative with per-line tridiagonal solves (Eq. 25-31, R4) against the oracle's
    whole-array-derivative assembly: right-hand side, RK4 steps, kick, batched slots."""
    g, o = both(cfg, batch=2)
    M = cfg["n_modes"]
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=6)
    g.import_state(X, replica=0); g.import_state(0.5 * X, replica=1); o.import_state(X)
    Fg, Fo = g.export_rhs(), o.rhs(X, via_deriv=True)
    assert rel_l2(Fg, Fo) < 1e-12
    g.step(3, cfg["dt"]); o.step(3, cfg["dt"])
    assert rel_l2(g.export_state(0), o.export_state()) < 1e-12
    assert rel_l2(2.0 * g.export_state(1), o.export_state()) < 1e-12
    gen = dict(c0=0.0, lin_q=[0.7, -0.4, 0.2][:M], quad=[[0.5, 0.2, -0.1][:M], [0.1, -0.3, 0.25][:M], [0.05, 0.15, 0.4][:M]][:M],
               lin_p=[0.0] * M)
    og, oo = make_obs(gpu_mod(), gen), make_obs(oracle, gen)
    g.import_state(X, replica=0); o.import_state(X)
    g.kick(og); o.kick(oo)
    assert rel_l2(g.export_state(0), o.export_state()) < 1e-12
    g.close()


def test_compact6_closed_form_response():
    """Pin P1 with the Pade scheme on the CUDA path: config 1 in the sqrt(W_eq) gauge reaches the Brownian-oscillator
    closed form to 2e-7 (5e-8 measured by the survey; the explicit CENTRAL4 scheme gives 3e-5 on the same grid)."""
    cfg = ci.config("cfg1", scheme="compact6")
    P = gpu_mod()
    g = P.CHFPE(cfg)
    mu_g, _ = obs_pair("mu", 1)
    g.equilibrate()
    R = g.response_1d(mu_g, mu_g, 5, 500, cfg["dt"])
    gold = [0.0, 0.4704830104, 0.7836581507, 0.8508220546, 0.6713837425]
    assert np.max(np.abs(-R - np.array(gold))) < 2e-7
    g.close()


def test_response_2d_shrunken_config5():
    """Config 5 protocol (A = mu, B = C = alpha, t1 replicas batched) on the 10^6 shrink of its model with 3 slots:
    as many steps as the oracle affords in about half a minute (3 t1 x 3 t2 delays, 18 oracle steps of 2e7 values)."""
    cfg = ci.config("cfg4s10")
    g, o = both(cfg, batch=3)
    mu_g, mu_o = obs_pair("mu", 3)
    al_g, al_o = obs_pair("alpha", 3)
    g.equilibrate(); o.equilibrate()
    t1, t2 = [0, 1, 3], [0, 2, 5]
    Rg = g.response_2d(mu_g, al_g, al_g, t1, t2, cfg["dt"])
    Ro = o.response_2d(mu_o, al_o, al_o, t1, t2, cfg["dt"])
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    g.close()


def test_response_2d_round_larger_than_the_results_buffer():
    """(batch - 1) * n2 > 65536 results: a round is clamped to the rows the device results buffer holds; without the
    clamp the overflow lands in the arrays that follow it (the state of slot 0, the t1 trajectory) and R2 is wrong."""
    cfg = ci.config("cfg2", nq=[8], np=[8], depth=1)
    n1, n2 = 300, 256
    P = gpu_mod()
    g = P.CHFPE(cfg, batch=290, guard_bytes=1 << 20)
    o = oracle.RefCHFPE(cfg)
    g.equilibrate(); o.equilibrate()
    (mu_g, mu_o), (al_g, al_o) = obs_pair("mu", 1), obs_pair("alpha", 1)
    t1, t2 = list(range(n1)), [0] * 200 + list(range(n2 - 200))      # 256 samples per row, 55 steps (oracle time)
    R = g.response_2d(mu_g, al_g, mu_g, t1, t2, cfg["dt"])
    assert g.guards_intact()
    Ro = o.response_2d(mu_o, al_o, mu_o, t1, t2, cfg["dt"])
    assert np.max(np.abs(R - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    g.close()


TERMINATOR = [
    ("m1_generic_w", ci.config("cfg2", nq=[37], np=[41], depth=3, gauge="w", closure="terminator")),
    ("m1_depth0", ci.config("cfg1", nq=[33], np=[29], depth=0, closure="terminator")),
    ("m1_c2", ci.config("cfg2", nq=[33], np=[29], depth=2, scheme="central2", closure="terminator")),
    ("m2_brick", ci.config("cfg3s", nq=[7, 9], depth=2, closure="terminator")),
    ("m3_generic", ci.config("cfg4s8", nq=[7, 8, 6], np=[8, 6, 9], depth=2, closure="terminator", mass=[1.0, 0.8, 1.2])),
    ("m3_cube8", ci.config("cfg4s8", nq=[6, 5, 7], closure="terminator")),
    ("m3_cube16", ci.config("cfg4", nq=[5, 5, 6], depth=2, closure="terminator")),
]


@pytest.mark.parametrize("name,cfg", TERMINATOR, ids=[c[0] for c in TERMINATOR])
def test_terminator_closure(name, cfg):
    """Row f4 (first half): terminator closure of the top hierarchy level (reading R23) on every stage-kernel family
    (cooperative / generic kernels evaluate it inside the right-hand side, the brick and bulk-copy kernels add it with
    k_terminator_add): right-hand side, steps and a batched 2D response against the oracle."""
    g, o = both(cfg, batch=2)
    M = cfg["n_modes"]
    levels = [sum(n) for n in o.elements()]
    X = ci.seeded_state(cfg, levels, seed=13)
    g.import_state(X); g.import_state(X, replica=1); o.import_state(X)
    Fg, Fo = g.export_rhs(1), o.rhs(X)
    assert rel_l2(Fg, Fo) < 1e-13
    for k in range(o.K):
        assert np.linalg.norm(Fg[k] - Fo[k]) <= 1e-13 * np.linalg.norm(Fo)
    plain = oracle.RefCHFPE(dict(cfg, closure="truncate"))
    assert rel_l2(plain.rhs(X), Fo) > 1e-3                       # the closure is not a no-op on this state
    g.step(3, cfg["dt"]); o.step(3, cfg["dt"])
    assert rel_l2(g.export_state(0), o.export_state()) < 1e-12
    assert rel_l2(g.export_state(1), o.export_state()) < 1e-12
    mu_g, mu_o = obs_pair("mu", M)
    al_g, al_o = obs_pair("alpha", M)
    g.equilibrate(); o.equilibrate()
    Rg = g.response_2d(mu_g, al_g, mu_g, [0, 2, 3], [0, 1, 4], cfg["dt"] * 5)
    Ro = o.response_2d(mu_o, al_o, mu_o, [0, 2, 3], [0, 1, 4], cfg["dt"] * 5)
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    g.close()


def test_terminator_depth0_kramers_closed_form_on_the_cuda_path():
    """The Kramers limit of the closure on the CUDA path itself: depth 0, harmonic mode, V' = 1 -> damped oscillator."""
    import math
    zeta = 0.5
    cfg = ci.config("cfg1", depth=0, gauge="w", closure="terminator")
    P = gpu_mod()
    g = P.CHFPE(cfg)
    g.equilibrate()
    mu = make_obs(P, ci.observable("mu", 1))
    R = g.response_1d(mu, mu, 21, 100, 1e-3)
    t = np.arange(21) * 0.1
    Om = math.sqrt(1.0 - zeta * zeta / 4.0)
    assert np.max(np.abs(-R - np.exp(-zeta * t / 2.0) * np.sin(Om * t) / Om)) < 1e-7
    g.close()


def test_terminator_rejected_where_it_is_not_implemented():
    P = gpu_mod()
    with pytest.raises(P.ChfpeError):
        P.CHFPE(ci.config("cfg1", scheme="compact6", closure="terminator"))
    with pytest.raises(P.ChfpeError):
        P.Hermite(ci.config("cfg1", np=[6], closure="terminator"))


def test_step_reports_divergence_from_the_call_that_diverged():
    """Norm guard of chfpe_step (SURVEY 8(b) errors): the literal W gauge is semi-discretely unstable on a (q,p) grid
    (reading R7; a config-2-like run reaches 1e30 by t = 3), so a propagation must return
    CHFPE_ERR_DIVERGED from the chfpe_step call in which the norm left its bound -- long before any value is
    non-finite -- while the default sqrt(W_eq) gauge runs through the same protocol untouched."""
    P = gpu_mod()
    base = dict(nq=[64], np=[64], depth=6, qmin=[-8.0], qmax=[8.0], pmin=[-8.0], pmax=[8.0])
    mu = make_obs(P, ci.observable("mu", 1))
    g = P.CHFPE(ci.config("cfg2", gauge="w", **base))
    g.equilibrate(); g.kick(mu)
    t_div = None
    for i in range(16):
        try:
            g.step(250, 1e-3)
        except P.ChfpeError as exc:
            assert "-4" in str(exc) or "diverg" in str(exc).lower(), exc
            t_div = 0.25 * (i + 1)
            break
    assert t_div is not None and t_div <= 3.0, t_div
    assert np.all(np.isfinite(g.export_state()))                 # caught on the norm, not on a NaN
    g.close()
    g = P.CHFPE(ci.config("cfg2", gauge="sqrt_eq", **base))
    g.equilibrate(); g.kick(mu)
    for i in range(16):
        g.step(250, 1e-3)
    g.close()


def test_response_2d_sharded_over_nccl_world1():
    """the multi-GPU path of the 2D response -- t1 rows round-robin over the ranks, one all_gather of
    n1 x n2 doubles -- with a CUDA engine and the NCCL backend (one rank: what a 1-GPU box can run; the row partition
    and the gather for world size 2 are covered on gloo in test_sharding_gloo.py).  Must equal the unsharded call."""
    import socket
    import torch
    import torch.distributed as dist
    from paper_2509_25840_b200 import sharding
    cfg = ci.config("cfg4s8", nq=[6, 6, 6], np=[6, 6, 6])
    g, o = both(cfg, batch=3)
    mu_g, _ = obs_pair("mu", 3)
    al_g, _ = obs_pair("alpha", 3)
    t1, t2 = [0, 2, 3, 7, 8], [0, 1, 4, 6]
    g.equilibrate()
    R_plain = g.response_2d(mu_g, al_g, al_g, t1, t2, cfg["dt"] * 10)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        g.equilibrate()
        R = sharding.response_2d_sharded(g, mu_g, al_g, al_g, t1, t2, cfg["dt"] * 10, device="cuda:0")
    finally:
        dist.destroy_process_group()
    assert R.shape == R_plain.shape and np.array_equal(R, R_plain)
    g.close()


class _LocalExchange:
    """Halo exchange between slab engines that live in ONE process (test only): plain device copies on the current
    stream, one slab after the other -- nothing waits on anything, so this is not a stand-in for several GPUs, only a
    check of the halo logic with the CUDA kernels."""

    def __init__(self, engines, geos):
        self.engines, self.geos = engines, geos

    def run_all(self, stage):
        from paper_2509_25840_b200 import sharding
        H = sharding.HALO
        views = [e.stage_input(stage) for e in self.engines]
        for r, (X, (lo, hi, hl, hh)) in enumerate(zip(views, self.geos)):
            n = X.shape[1]
            if hl:
                Y, (_, _, hl2, hh2) = views[r - 1], self.geos[r - 1]
                X[:, :hl] = Y[:, Y.shape[1] - hh2 - H:Y.shape[1] - hh2]
            if hh:
                Y, (_, _, hl2, hh2) = views[r + 1], self.geos[r + 1]
                X[:, n - hh:] = Y[:, hl2:hl2 + H]


@pytest.mark.parametrize("name,cfg,world", [("m3_tma", ci.config("cfg4s8", nq=[11, 5, 6]), 2),
                                            ("m3_tma_3slabs", ci.config("cfg4", nq=[13, 5, 5], depth=1), 3),
                                            ("m2_brick", ci.config("cfg3s", nq=[10, 7], depth=2), 2)])
def test_slab_decomposition_on_the_cuda_path(name, cfg, world):
    """Row f4 (second half), CUDA path: the grid is cut along q_1 into `world` slabs with two halo planes per inner face
    (sharding.slab_config); each slab is an ordinary CHFPE handle stepped stage by stage (chfpe_rk4_stage) with the
    halo planes of the stage input (chfpe_stage_input views) refreshed before every stage.  Owned planes must equal
    the undecomposed propagation and the oracle.  All slabs run in one process on one stream, one after the other."""
    from paper_2509_25840_b200 import sharding
    P = gpu_mod()
    g, o = both(cfg)
    X = ci.seeded_state(cfg, [sum(n) for n in o.elements()], seed=31)
    g.import_state(X); o.import_state(X)
    g.step(2, cfg["dt"]); o.step(2, cfg["dt"])
    want = g.export_state()
    assert rel_l2(want, o.export_state()) < 1e-12
    locs = [sharding.slab_config(cfg, r, world) for r in range(world)]
    engines = [P.CHFPE(lc, batch=1) for lc, _ in locs]
    geos = [ge for _, ge in locs]
    for e, (lo, hi, hl, hh) in zip(engines, geos):
        e.import_state(np.ascontiguousarray(X[:, lo - hl:hi + hh]))
    ex = _LocalExchange(engines, geos)
    for _ in range(2):
        for stage in range(4):
            ex.run_all(stage)
            for e in engines:
                e.rk4_stage(stage, cfg["dt"])
    got = np.concatenate([e.export_state()[:, hl:e.shape[0] - hh] for e, (lo, hi, hl, hh) in zip(engines, geos)], axis=1)
    assert got.shape == want.shape
    assert rel_l2(got, want) < 1e-13
    assert rel_l2(got, o.export_state()) < 1e-12
    # partial expectations over the owned planes add up to the global one
    al_g, al_o = obs_pair("alpha", cfg["n_modes"])
    props = [sharding.SlabPropagator(e, ge, None) for e, ge in zip(engines, geos)]
    tot = sum(p.expect_partial(al_g) for p in props)
    assert abs(tot - o.expect(al_o)) <= 1e-12 * max(1.0, abs(o.expect(al_o)))
    for e in engines:
        e.close()
    g.close()


def test_slab_propagator_over_nccl_world1_and_stage_api():
    """chfpe_rk4_stage x 4 == chfpe_step, and SlabPropagator + DistExchange on NCCL with one rank (the whole domain is
    one slab, no neighbours) equals the plain step bit for bit."""
    import socket
    import torch
    import torch.distributed as dist
    from paper_2509_25840_b200 import sharding
    cfg = ci.config("cfg4s8", nq=[6, 5, 7])
    P = gpu_mod()
    g, o = both(cfg)
    X = ci.seeded_state(cfg, [sum(n) for n in o.elements()], seed=5)
    g.import_state(X)
    g.step(2, cfg["dt"])
    want = g.export_state()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        loc, geo = sharding.slab_config(cfg, 0, 1)
        assert loc["nq"] == cfg["nq"] and geo == (0, cfg["nq"][0], 0, 0)
        e = P.CHFPE(loc)
        e.import_state(X)
        sharding.SlabPropagator(e, geo, sharding.DistExchange()).step(2, cfg["dt"])
        assert np.array_equal(e.export_state(), want)
        e.close()
    finally:
        dist.destroy_process_group()
    g.close()


def test_long_q3_line_falls_back_to_the_brick_kernel():
    """k_stage_tma tabulates dU/dq_s of a q_3 line in shared memory for lines of up to 64 bricks; longer lines must
    take the brick kernel (and still match the oracle)."""
    cfg = ci.config("cfg4s8", nq=[5, 5, 70], depth=1)
    g, o = both(cfg)
    assert g.stage_kernel() == "brick"
    X = ci.seeded_state(cfg, [sum(n) for n in o.elements()], seed=8)
    g.import_state(X); o.import_state(X)
    assert rel_l2(g.export_rhs(), o.rhs(X)) < 1e-13
    g.close()
    g64, o64 = both(ci.config("cfg4s8", nq=[5, 5, 64], depth=1))
    assert g64.stage_kernel() == "tma"
    X = ci.seeded_state(g64.cfg if hasattr(g64, "cfg") else ci.config("cfg4s8", nq=[5, 5, 64], depth=1), [sum(n) for n in o64.elements()], seed=8)
    g64.import_state(X); o64.import_state(X)
    assert rel_l2(g64.export_rhs(), o64.rhs(X)) < 1e-13
    g64.step(2, 1e-3); o64.step(2, 1e-3)
    assert rel_l2(g64.export_state(), o64.export_state()) < 1e-12
    g64.close()

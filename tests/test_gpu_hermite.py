"""Row f1: parity of the CUDA Hermite-representation path (chfpe_hermite_* through the C-ABI binding) with the numpy
oracle oracle/hermite.py on the same seeded inputs.  Tolerances as for the grid path (BASELINE.json north_star):
one right-hand side / kick 1e-13 relative L2, per-step 1e-12, response functions 1e-8 relative max."""
import os

import numpy as np
import pytest

import chfpe_inputs as ci
from oracle import hermite
from conftest import make_obs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def P():
    import paper_2509_25840_b200 as mod
    return mod


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def both(cfg, batch=1):
    return P().Hermite(cfg, batch=batch), hermite.RefHermite(cfg)


def gobs(d):
    return make_obs(P(), d)


def p_obs(M):
    """an observable with every coefficient non-zero, incl. the linear-momentum part"""
    return dict(c0=0.3, lin_q=[1.0, -0.7, 0.4][:M], quad=[[0.5, 0.2, -0.1][:M], [0.3, -0.4, 0.25][:M], [0.15, 0.1, 0.6][:M]][:M],
                lin_p=[0.8, -0.5, 0.3][:M])


SMALL = [
    ("m1", ci.config("cfg2", nq=[37], np=[9], depth=5)),
    ("m1_c2_mass", ci.config("cfg2", nq=[300], np=[4], depth=3, scheme="central2", mass=[1.3])),   # 2 CTAs per slab, ragged
    ("m1_kp1", ci.config("cfg2", nq=[21], np=[1], depth=2)),                                      # no Hermite neighbours at all
    ("m1_depth0", ci.config("cfg2", nq=[21], np=[5], depth=0)),                                   # a single element
    ("m2", ci.config("cfg3s", nq=[13, 11], np=[4, 5], depth=3)),
    ("m2_ragged_ctas", ci.config("cfg3s", nq=[40, 37], np=[3, 2], depth=2, mass=[1.0, 1.3])),      # 1480 q-points: 6 CTAs per slab
    ("m2_c2", ci.config("cfg3s", nq=[9, 10], np=[2, 6], depth=2, scheme="central2")),
    ("m3", ci.config("cfg4s8", nq=[7, 8, 6], np=[3, 2, 4], depth=3)),
    ("m3_ragged", ci.config("cfg4s8", nq=[11, 9, 13], np=[3, 4, 2], depth=2, mass=[1.0, 0.8, 1.2])),
    ("m3_kp1_mid", ci.config("cfg4s8", nq=[6, 5, 7], np=[3, 1, 2], depth=2, scheme="central2")),
    # the paper's compact (Pade) q-derivative: one Thomas line solve per slab, mode and q-line
    ("m1_compact6", ci.config("cfg2", nq=[67], np=[6], depth=4, scheme="compact6")),
    ("m1_compact6_256", ci.config("cfg2", nq=[256], np=[3], depth=2, scheme="compact6", mass=[1.3])),   # longest line
    ("m2_compact6", ci.config("cfg3s", nq=[23, 14], np=[3, 4], depth=2, scheme="compact6", mass=[1.0, 1.3])),
    ("m3_compact6", ci.config("cfg4s8", nq=[9, 12, 7], np=[3, 2, 3], depth=2, scheme="compact6")),
    ("m2_compact6_contig64", ci.config("cfg3s", nq=[70, 40], np=[2, 3], depth=1, scheme="compact6")),   # 64-line tiles, ragged
    ("m3_compact6_5pt", ci.config("cfg4s8", nq=[5, 6, 5], np=[2, 2, 2], depth=3, scheme="compact6")),  # shortest lines
]


@pytest.mark.parametrize("name,cfg", SMALL, ids=[c[0] for c in SMALL])
def test_rhs_step_kick_expect(name, cfg):
    g, o = both(cfg)
    M = cfg["n_modes"]
    assert g.K == o.K and g.shape == o.shape
    levels = [sum(n) for n in o.elems]
    X = ci.seeded_hermite_state(cfg, levels, seed=11)
    g.import_state(X); o.import_state(X)
    assert np.array_equal(g.export_state(), X)
    assert rel_l2(g.export_rhs(), o.rhs(o.c)) < 1e-13
    # expectations: polynomial in q plus <p_s> (from the k = e_s coefficients), on element 0 and on the last element
    d = p_obs(M)
    for el in (0, o.K - 1):
        ref = o.expect(d, element=el)
        got = g.expect(gobs(d), element=el)[0]
        assert abs(got - ref) <= 1e-13 * max(abs(ref), 1e-3), (el, got, ref)
    # RK4: the Horner form of the CUDA path against the textbook k1..k4 form of the oracle
    g.step(3, cfg["dt"]); o.step(3, cfg["dt"])
    assert rel_l2(g.export_state(), o.export_state()) < 1e-12
    # kick with a bilinear observable (every dX/dq_s depends on every q)
    g.kick(gobs(d)); o.kick(d)
    assert rel_l2(g.export_state(), o.export_state()) < 1e-13


@pytest.mark.parametrize("var,val", [("CHFPE_HERMITE_KC", "0"), ("CHFPE_HERMITE_KC", "4"), ("CHFPE_HERMITE_KC", "8"),
                                     ("CHFPE_HERMITE_PATCH", "44"), ("CHFPE_HERMITE_PATCH", "42"),
                                     ("CHFPE_HERMITE_PATCH", "24"), ("CHFPE_HERMITE_PATCH", "22"),
                                     ("CHFPE_HERMITE_PATCH", "0"), ("CHFPE_HERMITE_PCOL", "0")])
def test_every_stage_kernel_variant(var, val, monkeypatch):
    """CHFPE_HERMITE_KC: 0 = one thread per value, 4 / 8 = column kernel with that many Hermite indices of the last
    mode per thread (columns longer and shorter than a chunk, ragged last chunks, kp = 1).  CHFPE_HERMITE_PATCH = "AB":
    patch kernel with A x B points of (q_1, q_2) per thread (ragged patches, axes shorter than a patch + halo);
    CHFPE_HERMITE_PCOL=0: one slab per CTA instead of a walk over the column of the last Hermite index."""
    monkeypatch.setenv(var, val)
    for cfg in (ci.config("cfg2", nq=[37], np=[11], depth=4),
                ci.config("cfg3s", nq=[40, 37], np=[3, 9], depth=2, mass=[1.0, 1.3]),
                ci.config("cfg4s8", nq=[7, 8, 6], np=[2, 3, 5], depth=3),
                ci.config("cfg4s8", nq=[6, 5, 7], np=[3, 2, 1], depth=2, scheme="central2")):
        g, o = both(cfg)
        X = ci.seeded_hermite_state(cfg, [sum(n) for n in o.elems], seed=4)
        g.import_state(X); o.import_state(X)
        assert rel_l2(g.export_rhs(), o.rhs(o.c)) < 1e-13
        g.step(2, cfg["dt"]); o.step(2, cfg["dt"])
        assert rel_l2(g.export_state(), o.export_state()) < 1e-12
        g.close()


def test_compact6_strided_kernel_on_the_contiguous_axis(monkeypatch):
    """CHFPE_HERMITE_CONTIG=0: the one-thread-per-line kernel also serves the contiguous q axis (the fallback for axes
    longer than 64 points or fewer than 64 lines)."""
    monkeypatch.setenv("CHFPE_HERMITE_CONTIG", "0")
    cfg = ci.config("cfg4s8", nq=[9, 12, 7], np=[3, 2, 3], depth=2, scheme="compact6")
    g, o = both(cfg)
    X = ci.seeded_hermite_state(cfg, [sum(n) for n in o.elems], seed=8)
    g.import_state(X); o.import_state(X)
    assert rel_l2(g.export_rhs(), o.rhs(o.c)) < 1e-13
    g.step(2, cfg["dt"]); o.step(2, cfg["dt"])
    assert rel_l2(g.export_state(), o.export_state()) < 1e-12


def test_zero_steps_and_batch_slots_are_independent():
    cfg = ci.config("cfg3s", nq=[12, 9], np=[3, 4], depth=2)
    g = P().Hermite(cfg, batch=3)
    o = hermite.RefHermite(cfg)
    levels = [sum(n) for n in o.elems]
    Xs = [ci.seeded_hermite_state(cfg, levels, seed=s) for s in (1, 2, 3)]
    for b, X in enumerate(Xs):
        g.import_state(X, replica=b)
    g.step(0, cfg["dt"])
    for b, X in enumerate(Xs):
        assert np.array_equal(g.export_state(b), X)
    g.step(2, cfg["dt"])                             # one launch per stage advances all three slots
    d = p_obs(2)
    got = g.expect(gobs(d))
    for b, X in enumerate(Xs):
        o.import_state(X); o.step(2, cfg["dt"])
        assert rel_l2(g.export_state(b), o.export_state()) < 1e-12
        assert abs(got[b] - o.expect(d)) <= 1e-13 * abs(o.expect(d))


def test_equilibrium_state_and_residual():
    for cfg in (ci.config("cfg2", nq=[64], np=[6], depth=3), ci.config("cfg4s8", nq=[9, 8, 7], np=[2, 3, 2], depth=2)):
        g, o = both(cfg, batch=2)
        rg, ro = g.equilibrate(), o.equilibrate()
        assert rel_l2(g.export_state(0), o.export_state()) < 1e-14
        assert np.array_equal(g.export_state(1), g.export_state(0))
        assert abs(rg - ro) <= 1e-10 * ro
        one = ci.observable("one", cfg["n_modes"])
        assert abs(g.expect(gobs(one))[0] - 1.0) < 1e-12
        g.close()


def test_response_1d_anharmonic_sl():
    """config-2 model (anharmonic, LL + SL), nonlinear dipole: 400 steps sampled every 20."""
    cfg = ci.config("cfg2", nq=[64], np=[12], depth=6)
    g, o = both(cfg)
    g.equilibrate(); o.equilibrate()
    al, d = ci.observable("alpha", 1), ci.observable("mu_nl", 1)
    Rg = g.response_1d(gobs(al), gobs(d), 21, 20, 1e-3)
    Ro = o.response_1d(al, d, 21, 20, 1e-3)
    assert np.max(np.abs(Ro)) > 0.1
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))


def test_response_1d_ten_thousand_steps():
    """north_star: response functions within 1e-8 relative max after 10^4 steps (harmonic config-1 model, small mesh)."""
    cfg = ci.config("cfg1", nq=[33], np=[4], depth=3, qmin=[-8.0], qmax=[8.0])
    g, o = both(cfg)
    g.equilibrate(); o.equilibrate()
    mu = ci.observable("mu", 1)
    Rg = g.response_1d(gobs(mu), gobs(mu), 11, 1000, 1e-3)
    Ro = o.response_1d(mu, mu, 11, 1000, 1e-3)
    assert np.max(np.abs(Ro)) > 0.3
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))


def test_response_1d_compact6_and_its_closed_form():
    """COMPACT6 on the CUDA path: parity of a sampled response with the oracle, and the Brownian-oscillator closed form
    (tests/golden/bo_response_cfg1.txt) to 1e-5 on a mesh (h = 0.5) where CENTRAL4 is only good to 7e-4."""
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "bo_response_cfg1.txt"))
    cfg = ci.config("cfg1", nq=[37], np=[6], depth=3, qmin=[-9.0], qmax=[9.0], scheme="compact6")
    g, o = both(cfg)
    g.equilibrate(); o.equilibrate()
    mu = ci.observable("mu", 1)
    Rg = g.response_1d(gobs(mu), gobs(mu), 5, 500, 1e-3)
    Ro = o.response_1d(mu, mu, 5, 500, 1e-3)
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    assert np.allclose(gold[:, 0], 0.5 * np.arange(1, 5))
    assert np.max(np.abs(-Rg[1:] - gold[:, 1])) < 1e-5
    cfg2 = ci.config("cfg3s", nq=[14, 12], np=[4, 3], depth=2, scheme="compact6")
    g2, o2 = both(cfg2, batch=3)
    g2.equilibrate(); o2.equilibrate()
    mu2, al2 = ci.observable("mu", 2), ci.observable("alpha", 2)
    R2g = g2.response_2d(gobs(mu2), gobs(al2), gobs(al2), [0, 4, 6], [0, 5], 5e-3)
    R2o = o2.response_2d(mu2, al2, al2, [0, 4, 6], [0, 5], 5e-3)
    assert np.max(np.abs(R2g - R2o)) <= 1e-8 * np.max(np.abs(R2o))


def test_response_1d_three_modes():
    cfg = ci.config("cfg4s8", nq=[10, 9, 8], np=[3, 3, 3], depth=2)
    g, o = both(cfg)
    g.equilibrate(); o.equilibrate()
    mu, al = ci.observable("mu", 3), ci.observable("alpha", 3)
    Rg = g.response_1d(gobs(al), gobs(al), 6, 10, 2e-3)
    Ro = o.response_1d(al, al, 6, 10, 2e-3)
    assert np.max(np.abs(Ro)) > 0.05
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    del mu


@pytest.mark.parametrize("batch", [2, 3, 5])
def test_response_2d_batched_over_t1(batch):
    """Eq. (16): rounds of batch-1 replicas (full, ragged and single rounds), repeated and zero delays."""
    cfg = ci.config("cfg3s", nq=[12, 11], np=[4, 3], depth=2)
    g, o = both(cfg, batch=batch)
    g.equilibrate(); o.equilibrate()
    mu, al = ci.observable("mu", 2), ci.observable("alpha", 2)
    t1, t2 = [0, 3, 3, 7, 12], [0, 4, 9]
    Rg = g.response_2d(gobs(mu), gobs(al), gobs(al), t1, t2, 5e-3)
    Ro = o.response_2d(mu, al, al, t1, t2, 5e-3)
    assert np.max(np.abs(Ro)) > 1e-3
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    assert np.array_equal(Rg[1], Rg[2])              # repeated t1 sample


@pytest.mark.parametrize("scheme", ["central4", "compact6"])
def test_protocols_on_the_march_kernel(scheme):
    """The 1D and batched 2D response drivers on a three-mode n_1 x 32 x 32 mesh, i.e. with k_hermite_stage_tma under them
    (explicit stencils: <CMP=false>; COMPACT6: <CMP=true> + the q_1 line pass): equilibrium state, kick, 40 RK4 steps with
    batch slots at different trajectory positions, expectation values, against the oracle's plain loops."""
    cfg = ci.config("cfg4h", nq=[6, 32, 32], np=[2, 2, 2], depth=1, scheme=scheme)
    g, o = both(cfg, batch=3)
    assert g.stage_kernel() == ("tma" if scheme == "central4" else "compact_tma")
    g.equilibrate(); o.equilibrate()
    mu, al = ci.observable("mu", 3), ci.observable("alpha", 3)
    R1g = g.response_1d(gobs(mu), gobs(mu), 9, 5, 4e-3)
    R1o = o.response_1d(mu, mu, 9, 5, 4e-3)
    assert np.max(np.abs(R1o)) > 1e-3
    assert np.max(np.abs(R1g - R1o)) <= 1e-8 * np.max(np.abs(R1o))
    g.equilibrate(); o.equilibrate()
    t1, t2 = [0, 4, 9], [0, 3, 8]
    Rg = g.response_2d(gobs(mu), gobs(al), gobs(al), t1, t2, 4e-3)
    Ro = o.response_2d(mu, al, al, t1, t2, 4e-3)
    assert np.max(np.abs(Ro)) > 1e-5
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    g.close()


@pytest.mark.parametrize("batch,n2", [(3, 2), (5, 3), (4, 1), (2, 1)])
def test_response_3d_batched(batch, n2):
    """Eq. (17): groups of (batch-1)/2 t1 samples (batch-1 for a single waiting time), ragged last group, repeated and
    zero delays, against the plain triple loop of the oracle."""
    cfg = ci.config("cfg3s", nq=[10, 9], np=[4, 3], depth=2, scheme="compact6" if batch == 5 else "central4")
    g, o = both(cfg, batch=batch)
    g.equilibrate(); o.equilibrate()
    mu, al, nl = ci.observable("mu", 2), ci.observable("alpha", 2), ci.observable("mu_nl", 2)
    t1, t2, t3 = [0, 2, 5], [1, 3, 3][:n2], [0, 2, 3]
    Rg = g.response_3d(gobs(mu), gobs(nl), gobs(al), gobs(nl), t1, t2, t3, 5e-2)
    Ro = o.response_3d(mu, nl, al, nl, t1, t2, t3, 5e-2)
    assert Rg.shape == (3, n2, 3) and np.max(np.abs(Ro)) > 1e-3
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))


def test_response_3d_needs_slots():
    cfg = ci.config("cfg2", nq=[16], np=[3], depth=1)
    g = P().Hermite(cfg, batch=2)
    g.equilibrate()
    mu = gobs(ci.observable("mu", 1))
    with pytest.raises(P().ChfpeError):
        g.response_3d(mu, mu, mu, mu, [0], [0, 1], [0], 1e-3)


@pytest.mark.parametrize("scheme", ["central4", "compact6"])
def test_no_entry_point_writes_outside_the_workspace(scheme, monkeypatch):
    """Canary bytes on both sides of the caller-owned workspace survive every entry point of every stage-kernel family
    (ragged meshes, all slots in use)."""
    for var, val in ((None, None), ("CHFPE_HERMITE_KC", "0"), ("CHFPE_HERMITE_KC", "8"), ("CHFPE_HERMITE_PATCH", "44"),
                     ("CHFPE_HERMITE_CONTIG", "0")):
        if var:
            monkeypatch.setenv(var, val)
        for cfg in (ci.config("cfg2", nq=[37], np=[5], depth=3, scheme=scheme),
                    ci.config("cfg4s8", nq=[9, 11, 7], np=[3, 2, 5], depth=2, scheme=scheme)):
            M = cfg["n_modes"]
            g = P().Hermite(cfg, batch=3, guard_bytes=1 << 16)
            mu, al = gobs(ci.observable("mu", M)), gobs(ci.observable("alpha", M))
            g.equilibrate(2, cfg["dt"])
            g.kick(mu); g.step(2, cfg["dt"]); g.expect(al); g.export_rhs(2)
            g.equilibrate()
            g.response_1d(mu, mu, 3, 2, cfg["dt"])
            g.equilibrate()
            g.response_2d(mu, al, al, [0, 1, 2], [0, 2], cfg["dt"])
            g.equilibrate()
            g.response_3d(mu, al, al, mu, [0, 1], [1, 2], [0, 1], cfg["dt"])
            g.import_state(g.export_state(1), replica=2)
            assert g.guards_intact(), (var, val, cfg["name"])
            g.close()
        if var:
            monkeypatch.delenv(var)


def test_closed_forms_on_the_cuda_path():
    """The pins of the oracle hold for the CUDA path on its own: Brownian-oscillator R1 (tests/golden/bo_response_cfg1.txt,
    literal Eq. 15 = -R_phys) and the 2D closed form 2 R_phys(t1) R_phys(t2) (tests/golden/r2_closed_form.txt)."""
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "bo_response_cfg1.txt"))
    cfg = ci.config("cfg1", nq=[73], np=[6], depth=3, qmin=[-9.0], qmax=[9.0])
    g = P().Hermite(cfg, batch=2)
    g.equilibrate()
    mu, al = gobs(ci.observable("mu", 1)), gobs(ci.observable("alpha", 1))
    steps = [int(round(t / 1e-3)) for t in gold[:, 0]]
    assert np.allclose(np.array(steps) * 1e-3, gold[:, 0], atol=1e-12)
    now, worst = 0, 0.0
    g.kick(mu)
    one = np.empty(1)
    for s, ref in zip(steps, gold[:, 1]):
        g.step(s - now, 1e-3); now = s
        worst = max(worst, abs(-g.expect(mu)[0] - ref))
    assert worst < 1e-4, worst
    g2 = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "r2_closed_form.txt"))
    g.equilibrate()
    R = g.response_2d(mu, al, mu, [int(round(g2[0] / 2e-3))], [int(round(g2[1] / 2e-3))], 2e-3)
    assert abs(R[0, 0] - g2[2]) < 2e-4
    del one



@pytest.mark.parametrize("kp,depth", [([2, 2, 2], 2), ([1, 1, 8], 1)], ids=["kp222_depth2", "kp118_depth1"])
def test_cube32_specialisation_up_to_the_mesh_edges(kp, depth):
    """The 32^3 compile-time specialisation of the patch kernel (`cube32` branch: lane-axis stencil on warp shuffles
    with zero row ends, 4 x 8 x 32 CTA tiles, immediate-offset ghost handling) with a state that is non-zero on every
    mesh face, edge and corner: right-hand side and two RK4 steps against oracle/hermite.py on the whole mesh, for the
    default launch shape and for CHFPE_HERMITE_TILE / _FIXED / _PCOL = 0.  kp = [1, 1, 8] walks a full column of the last
    Hermite index (the column walk of the bench configuration), kp = [2, 2, 2] exercises every Hermite neighbour."""
    cfg = ci.config("cfg4h", np=kp, depth=depth)
    assert cfg["nq"] == [32, 32, 32]
    o = hermite.RefHermite(cfg)
    X = ci.seeded_hermite_state(cfg, [sum(n) for n in o.elems], seed=9)
    # the seeded envelope exp(-q.q/4) is 1e-4 at the faces; lift the faces to O(1) so that a ghost or wrap-around bug
    # there cannot hide below the tolerance
    rng = np.random.default_rng(17)
    X = X + 0.05 * rng.uniform(-1.0, 1.0, size=X.shape)
    for i in (0, 1, 30, 31):
        assert np.abs(X[..., i, :, :]).max() > 1e-2 and np.abs(X[..., :, i, :]).max() > 1e-2 and np.abs(X[..., :, :, i]).max() > 1e-2
    Fo = o.rhs(X)
    o.import_state(X)
    o.step(2, cfg["dt"])
    Yo = o.export_state()
    for var in ("tma", None, "CHFPE_HERMITE_TILE", "CHFPE_HERMITE_FIXED", "CHFPE_HERMITE_PCOL"):
        # "tma": the default on this mesh, the bulk-copy march kernel; the others: the patch kernel and its launch shapes
        if var != "tma":
            os.environ["CHFPE_HERMITE_TMA"] = "0"
            if var:
                os.environ[var] = "0"
        try:
            g = P().Hermite(cfg)
        finally:
            if var != "tma":
                del os.environ["CHFPE_HERMITE_TMA"]
                if var:
                    del os.environ[var]
        assert g.stage_kernel() == ("tma" if var == "tma" else "patch")
        g.import_state(X)
        F = g.export_rhs()
        assert rel_l2(F, Fo) < 1e-13, var
        for sl in (np.s_[..., 0:2, :, :], np.s_[..., 30:32, :, :], np.s_[..., :, 0:2, :], np.s_[..., :, 30:32, :],
                   np.s_[..., :, :, 0:2], np.s_[..., :, :, 30:32]):   # the faces on their own
            assert np.linalg.norm(F[sl] - Fo[sl]) <= 1e-13 * np.linalg.norm(Fo[sl]), (var, sl)
        g.step(2, cfg["dt"])
        assert rel_l2(g.export_state(), Yo) < 1e-12, var
        g.close()


MARCH = [
    ("ten_planes", dict(nq=[10, 32, 32], np=[2, 2, 2], depth=2)),                 # an odd number of bands, every neighbour kind
    ("six_planes_c2", dict(nq=[6, 32, 32], np=[2, 1, 3], depth=2, scheme="central2", mass=[1.0, 0.8, 1.2])),
    ("depth0_long", dict(nq=[70, 32, 32], np=[1, 2, 2], depth=0)),                # no hierarchy neighbours, 35 bands
    ("kp1", dict(nq=[8, 32, 32], np=[1, 1, 1], depth=3)),                         # no Hermite neighbours: couplings only
    # COMPACT6: the march kernel solves the Pade derivative along q_2 and q_3 itself, a line pass adds the q_1 part
    ("compact6", dict(nq=[8, 32, 32], np=[2, 2, 2], depth=2, scheme="compact6", mass=[1.0, 0.8, 1.2])),
    ("compact6_cube32", dict(nq=[32, 32, 32], np=[2, 1, 2], depth=1, scheme="compact6")),   # q_1 pass with the line in registers
]


@pytest.mark.parametrize("name,kw", MARCH, ids=[c[0] for c in MARCH])
def test_march_kernel_on_other_mesh_lengths(name, kw, monkeypatch):
    """k_hermite_stage_tma (bulk-copy march along q_1 in bands of two planes) on n_1 x 32 x 32 meshes: three bands (the
    shortest mesh the path accepts has six planes), an odd number of bands, more bands than the ring has parities, absent kinds of every sort.  The state is O(1) on every
    mesh face.  Right-hand side (a = 0: y is not read), three RK4 steps (the last stage writes y in place) and two
    batch slots against the oracle; CHFPE_HERMITE_TMA=0 must give the patch kernel's result on the same input."""
    cfg = ci.config("cfg4h", **kw)
    g, o = both(cfg, batch=2)
    compact = cfg["scheme"] == "compact6"
    assert g.stage_kernel() == ("compact_tma" if compact else "tma")
    X = ci.seeded_hermite_state(cfg, [sum(n) for n in o.elems], seed=21)
    X = X + 0.05 * np.random.default_rng(3).uniform(-1.0, 1.0, size=X.shape)
    g.import_state(X); g.import_state(2.0 * X, replica=1); o.import_state(X)
    Fo = o.rhs(o.c)
    assert rel_l2(g.export_rhs(), Fo) < 1e-13
    assert rel_l2(g.export_rhs(replica=1), 2.0 * Fo) < 1e-13
    g.step(3, cfg["dt"]); o.step(3, cfg["dt"])
    Yo = o.export_state()
    assert rel_l2(g.export_state(), Yo) < 1e-12
    assert rel_l2(g.export_state(replica=1), 2.0 * Yo) < 1e-12
    monkeypatch.setenv("CHFPE_HERMITE_TMA", "0")
    p = P().Hermite(cfg)
    assert p.stage_kernel() == ("compact" if compact else "patch")
    p.import_state(X)
    assert rel_l2(p.export_rhs(), Fo) < 1e-13
    n0 = p.launch_count(); p.step(1, cfg["dt"])
    assert p.launch_count() - n0 == (16 if compact else 4)   # COMPACT6 without the march kernel: pointwise pass + three line passes
    n0 = g.launch_count(); g.step(1, cfg["dt"])
    assert g.launch_count() - n0 == (8 if compact else 4)    # with it: fused kernel + the q_1 line pass
    p.close(); g.close()


@pytest.mark.parametrize("scheme", ["central4", "compact6"])
def test_march_kernel_is_bitwise_reproducible_at_full_size(scheme):
    """The march kernel synchronises its warps with mbarriers only (ring slots, exchange planes, the COMPACT6 line solves):
    a missing wait would show up as a race, i.e. as run-to-run differences, most likely with all 10240 CTAs of the bench
    workload in flight.  The kernel has no atomics and a fixed summation order, so two runs from the same state must agree
    BITWISE: right-hand side twice, then two RK4 steps from the same state twice (the last stage updates y in place)."""
    cfg = ci.config("cfg4h", scheme=scheme)
    if torch.cuda.mem_get_info()[0] < 20e9:
        pytest.skip("needs 20 GB of device memory")
    g = P().Hermite(cfg)
    assert g.stage_kernel() == ("tma" if scheme == "central4" else "compact_tma")
    gen = torch.Generator(device="cuda").manual_seed(5)
    X = torch.rand(g.shape, dtype=torch.float64, device="cuda", generator=gen) - 0.5
    g.import_state(X)
    F1 = g.export_rhs_device().clone()
    F2 = g.export_rhs_device()
    assert torch.equal(F1, F2)
    assert bool(torch.isfinite(F1).all()) and float(F1.abs().max()) > 0.0
    del F1, F2
    g.step(2, cfg["dt"])
    Y1 = g.export_state_device()
    g.import_state(X)
    g.step(2, cfg["dt"])
    Y2 = g.export_state_device()
    assert torch.equal(Y1, Y2)
    g.close()


def test_full_size_rhs_on_an_embedded_block():
    """The bench workload (cfg4h: 32^3 q mesh, 8^3 Hermite functions, 20 elements = 3.36e8 values, launch configuration
    of bench.py --representation hermite).  The state is zero outside a 9 x 10 x 11 block of the q mesh; zero ghosts
    (R9) make the right-hand side inside the block equal to that of the oracle on the block alone (same mesh width,
    shifted origin), for every element and every Hermite index."""
    cfg = ci.config("cfg4h")
    if torch.cuda.mem_get_info()[0] < 12e9:
        pytest.skip("needs 12 GB of device memory")
    off, ext = (5, 14, 19), (9, 10, 11)
    h = [(cfg["qmax"][s] - cfg["qmin"][s]) / (cfg["nq"][s] - 1) for s in range(3)]
    sub = ci.config("cfg4h", nq=list(ext), qmin=[cfg["qmin"][s] + h[s] * off[s] for s in range(3)],
                    qmax=[cfg["qmin"][s] + h[s] * (off[s] + ext[s] - 1) for s in range(3)])
    o = hermite.RefHermite(sub)
    assert max(abs(o.h[s] - h[s]) for s in range(3)) < 1e-14
    Xs = ci.seeded_hermite_state(sub, [sum(n) for n in o.elems], seed=5)
    g = P().Hermite(cfg)
    X = torch.zeros(g.shape, dtype=torch.float64, device="cuda")
    blk = (slice(None),) * 4 + tuple(slice(off[s], off[s] + ext[s]) for s in range(3))
    X[blk] = torch.from_numpy(Xs).cuda()
    g.import_state(X)
    F = g.export_rhs_device()[blk].cpu().numpy()
    Fo = o.rhs(Xs)
    assert rel_l2(F, Fo) < 1e-13
    assert g.stage_kernel() == "tma"
    for var in ("CHFPE_HERMITE_TMA", "CHFPE_HERMITE_TILE", "CHFPE_HERMITE_FIXED", "CHFPE_HERMITE_PCOL"):   # the patch kernel's launch shapes at this size
        os.environ[var] = "0"
        os.environ["CHFPE_HERMITE_TMA"] = "0"
        try:
            g2 = P().Hermite(cfg)
        finally:
            del os.environ["CHFPE_HERMITE_TMA"]
            if var != "CHFPE_HERMITE_TMA":
                del os.environ[var]
        assert g2.stage_kernel() == "patch"
        g2.import_state(X)
        assert rel_l2(g2.export_rhs_device()[blk].cpu().numpy(), Fo) < 1e-13, var
        g2.close()
    del X
    # one RK4 step at full size is four launches of the stage kernel and nothing else
    n0 = g.launch_count()
    g.step(1, cfg["dt"])
    assert g.launch_count() - n0 == 4
    g.close()


def test_response_2d_round_larger_than_the_results_buffer():
    """(batch - 1) * n2 > 65536 results: a round must be clamped to the rows the device results buffer holds (the
    Hermite results region is the last carve of the workspace: an overflow would land outside it)."""
    cfg = ci.config("cfg2", nq=[9], np=[3], depth=1)
    n1, n2 = 300, 256
    g = P().Hermite(cfg, batch=290, guard_bytes=1 << 20)
    o = hermite.RefHermite(cfg)
    g.equilibrate(); o.equilibrate()
    mu_d, al_d = ci.observable("mu", 1), ci.observable("alpha", 1)
    t1, t2 = list(range(n1)), [0] * 200 + list(range(n2 - 200))      # 256 samples per row, 55 steps (oracle time)
    R = g.response_2d(gobs(mu_d), gobs(al_d), gobs(mu_d), t1, t2, cfg["dt"])
    assert g.guards_intact()
    Ro = o.response_2d(mu_d, al_d, mu_d, t1, t2, cfg["dt"])
    assert np.max(np.abs(R - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    g.close()

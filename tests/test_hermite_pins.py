"""Pins of the Hermite-representation oracle (oracle/hermite.py, row f1): the closed-form Brownian-oscillator response
with fourth-order convergence in the q mesh, the exact first-moment ODE (incl. <p> from the k = 1 coefficient), and
cross-validation against the independent phase-space-grid oracle (oracle/chfpe_ref.c) on anharmonic models with LL+SL
coupling for one and two modes.  CPU only."""
import numpy as np
import scipy.linalg

import chfpe_inputs as ci
import oracle
from oracle import hermite
from conftest import make_obs

ONE = {"c0": 1.0, "lin_q": [0.0] * 3, "quad": [[0.0] * 3] * 3, "lin_p": [0.0] * 3}


def bo_matrix(w0=1.0, zeta=0.5, gamma=1.0):
    return np.array([[0, 1, 0], [-w0 ** 2, 0, 1], [0, -zeta * gamma, -gamma]], dtype=float)


def harmonic(n, half=9.0, kp=8, depth=3):
    return ci.config("cfg1", nq=[n], np=[kp], depth=depth, qmin=[-half], qmax=[half])


def test_element_order_matches_the_grid_oracle():
    for M, depth, name in ((1, 5, "cfg1"), (2, 4, "cfg3s"), (3, 3, "cfg4s8")):
        g = oracle.RefCHFPE(ci.config(name, nq=[5] * M, np=[5] * M, depth=depth))
        assert hermite.enumerate_elements(M, depth) == [tuple(n) for n in g.elements()]


def test_closed_form_response_converges_at_fourth_order():
    """Literal Eq. (15) = -R_phys(t) = -[e^{At}]_{01}; the only error is the q stencil (h^4): the Hermite and hierarchy
    truncations are exact for first moments of the harmonic + LL model."""
    mu = ci.observable("mu", 1)
    exact = scipy.linalg.expm(0.5 * bo_matrix())[0, 1]
    errs = []
    for n in (37, 73):                                           # h = 0.5, 0.25 on [-9, 9]
        o = hermite.RefHermite(harmonic(n))
        res = o.equilibrate()
        assert abs(o.expect(ONE) - 1.0) < 1e-12
        R = o.response_1d(mu, mu, 2, 500, 1e-3)
        assert R[0] == 0.0
        errs.append(abs(-R[1] - exact))
        assert res < (2e-3 if n == 37 else 2e-4)                 # equilibrium is stationary up to the stencil error
    assert 12.0 < errs[0] / errs[1] < 20.0 and errs[1] < 3e-5


def test_first_moments_and_bath_force():
    """<q>, <p> (from c_{k=1}) and <Omega> = -int W^(1) (from element 1) obey the 3 x 3 linear ODE of pin P3."""
    o = hermite.RefHermite(harmonic(73))
    o.equilibrate()
    o.kick(ci.observable("mu", 1))
    o.step(400, 1e-3)
    y = scipy.linalg.expm(0.4 * bo_matrix()) @ np.array([0.0, -1.0, 0.0])
    q = {"c0": 0.0, "lin_q": [1.0], "quad": [[0.0]], "lin_p": [0.0]}
    p = {"c0": 0.0, "lin_q": [0.0], "quad": [[0.0]], "lin_p": [1.0]}
    got = [o.expect(q), o.expect(p), -o.expect(ONE, element=1)]
    assert np.max(np.abs(np.array(got) - y)) < 3e-5
    assert abs(y[1]) > 0.5 and abs(y[2]) > 0.05                  # all three are exercised


def test_two_dimensional_closed_form():
    """Pin P4 on the Hermite oracle: R2_lib(t2, t1) = 2 R_phys(t1) R_phys(t2) for A = C = q, B = q^2 on the harmonic
    + LL model (tests/golden/r2_closed_form.txt, literal Eq. 16), zero for a linear B; second moments of the
    harmonic model stay within Hermite index 2 and hierarchy level 2, so only the q stencil limits it."""
    import os
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "r2_closed_form.txt"))
    mu, al = ci.observable("mu", 1), ci.observable("alpha", 1)
    errs = []
    for n in (37, 73):                                           # h = 0.5, 0.25: the stencil error falls as h^4
        o = hermite.RefHermite(harmonic(n, kp=6, depth=3))
        o.equilibrate()
        R = o.response_2d(mu, al, mu, [0, int(round(gold[0] / 2e-3))], [0, int(round(gold[1] / 2e-3))], 2e-3)
        errs.append((abs(R[1, 1] - gold[2]), abs(R[0, 1])))
        assert R[1, 0] == 0.0                                    # the B kick empties k = 0
    assert errs[1][0] < 2e-4 and 10.0 < errs[0][0] / errs[1][0] < 22.0 and abs(gold[2]) > 1.0
    assert errs[1][1] < 2e-4 and errs[0][1] / errs[1][1] > 10.0  # R_phys(t1 = 0) = 0 up to the stencil error
    o.equilibrate()
    R0 = o.response_2d(mu, mu, mu, [400], [600], 2e-3)
    assert abs(R0[0, 0]) < 1e-7


def test_cross_validation_with_the_grid_oracle_one_mode():
    """Anharmonic U, LL + SL coupling, nonlinear dipole, kick by alpha = q^2: two independent discretisations of
    Eq. (8) (Hermite functions vs a momentum mesh, numpy vs C) agree to the stencil error of either."""
    al, d = ci.observable("alpha", 1), ci.observable("mu_nl", 1)
    oh = hermite.RefHermite(ci.config("cfg2", nq=[64], np=[20], depth=6))
    oh.equilibrate()
    Rh = oh.response_1d(al, d, 2, 500, 1e-3)
    og = oracle.RefCHFPE(ci.config("cfg2", nq=[64], np=[64], depth=6))
    og.equilibrate()
    Rg = og.response_1d(make_obs(oracle, al), make_obs(oracle, d), 2, 500, 1e-3)
    assert np.max(np.abs(Rh)) > 0.2
    assert np.max(np.abs(Rh - Rg)) < 1e-4


def test_cross_validation_with_the_grid_oracle_two_modes():
    """Two coupled anharmonic modes (cross term q1^2 q2), both baths: mode indices, couplings and the kick of both
    modes against the grid oracle (coarse meshes)."""
    al, d = ci.observable("alpha", 2), ci.observable("mu_nl", 2)
    oh = hermite.RefHermite(ci.config("cfg3s", nq=[22, 22], np=[7, 7], depth=2))
    oh.equilibrate()
    Rh = oh.response_1d(al, d, 2, 60, 5e-3)
    og = oracle.RefCHFPE(ci.config("cfg3s", nq=[22, 22], np=[22, 22], depth=2))
    og.equilibrate()
    Rg = og.response_1d(make_obs(oracle, al), make_obs(oracle, d), 2, 60, 5e-3)
    assert abs(Rh[1]) > 0.3 and abs(Rh[1] - Rg[1]) < 8e-3 * abs(Rg[1])   # h = 0.57 meshes: 0.4 % apart


def test_truncations_are_zero_ghosts():
    """A state living in the top Hermite index and top hierarchy level only couples downwards."""
    cfg = ci.config("cfg2", nq=[12], np=[4], depth=2)
    o = hermite.RefHermite(cfg)
    c = np.zeros(o.shape)
    c[2, 3, :] = np.exp(-o.q[0] ** 2)                            # top level, top Hermite index
    F = o.rhs(c)
    # element 1 would receive it as c^(n+e)_{k-1} at k = 4 (outside), the level above does not exist
    assert np.all(F[0] == 0.0) and np.all(F[1] == 0.0)
    assert np.any(F[2, 2] != 0.0) and np.all(F[2, :2] == 0.0)
    assert np.allclose(F[2, 3], -2.0 * cfg["gamma"][0] * c[2, 3], rtol=1e-15, atol=0)
    c[:] = 0.0
    c[1, 0, :] = np.exp(-o.q[0] ** 2)                            # level 1, k = 0: feeds level 0 at k = 1 only (Phi lowers n, raises k)
    F = o.rhs(c)
    assert np.any(F[0, 1] != 0.0) and np.all(F[0, 0] == 0.0) and np.all(F[0, 2:] == 0.0) and np.all(F[2] == 0.0)


def test_compact6_derivative_is_sixth_order_and_matches_the_c_oracle():
    """The Pade q-derivative of the Hermite oracle (scipy banded solve): order 6 on a Gaussian (ratio 64 when h halves;
    the printed a = 7/18 would not even be consistent, R4), and the same numbers as the independent Thomas recurrence
    of oracle/chfpe_ref.c on a random vector (truncated matrices, R9), along the first and the last q axis."""
    errs = []
    for n in (33, 65):
        o = hermite.RefHermite(ci.config("cfg3s", nq=[n, 7], np=[1, 1], depth=0, scheme="compact6",
                                         qmin=[-8.0, -6.0], qmax=[8.0, 6.0]))
        x = o.q[0]
        g = (np.exp(-0.5 * x ** 2)[:, None] * np.ones(7)[None, :]).reshape(1, 1, n, 7)
        errs.append(np.max(np.abs(o.dq(g, 0) + x[None, None, :, None] * g)))
    assert 45.0 < errs[0] / errs[1] < 100.0 and errs[1] < 1e-5
    rng = np.random.default_rng(3)
    for nq, axis in (([19, 8], 0), ([6, 23], 1)):
        o = hermite.RefHermite(ci.config("cfg3s", nq=nq, np=[2, 1], depth=0, scheme="compact6"))
        g = rng.standard_normal((2, 1) + tuple(nq))
        d = o.dq(g, axis)
        # the C oracle differentiates a phase-space array along one of its axes: use a 1-mode grid whose q axis is the line
        n = nq[axis]
        oc = oracle.RefCHFPE(ci.config("cfg1", nq=[n], np=[5], depth=0, scheme="compact6", qmin=[o.q[axis][0]],
                                       qmax=[o.q[axis][-1]]))
        lines = np.moveaxis(g, 2 + axis, -1).reshape(-1, n)
        ref = np.empty_like(lines)
        for i, line in enumerate(lines):
            f = np.repeat(line[:, None], 5, axis=1)                # constant along p: every column is the same line
            ref[i] = oc.deriv_axis(f, 0)[:, 2]
        got = np.moveaxis(d, 2 + axis, -1).reshape(-1, n)
        assert np.max(np.abs(got - ref)) < 1e-12 * np.max(np.abs(ref))


def test_compact6_closed_form_response():
    """Brownian-oscillator R1 with the paper's scheme: at h = 0.5 the compact derivative is an order of magnitude closer
    to the closed form than CENTRAL4, and the error falls by far more than 16 when h halves."""
    mu = ci.observable("mu", 1)
    exact = scipy.linalg.expm(0.5 * bo_matrix())[0, 1]
    err = {}
    for scheme, n in (("central4", 37), ("compact6", 37), ("compact6", 73)):
        o = hermite.RefHermite(dict(harmonic(n), scheme=scheme))
        o.equilibrate()
        R = o.response_1d(mu, mu, 2, 500, 1e-3)
        err[(scheme, n)] = abs(-R[1] - exact)
    assert err[("compact6", 37)] < 0.1 * err[("central4", 37)]
    assert err[("compact6", 73)] < err[("compact6", 37)] / 30.0 or err[("compact6", 73)] < 1e-9


def test_third_order_closed_forms():
    """Pin P4b on the Hermite oracle (Eq. 17, harmonic + LL model, c = R_phys): A = D = q, B = C = q^2 gives
    -4 c(t1) c(t2) c(t3); A = B = q, C = D = q^2 gives -4 c(t3) [c(t2) c(t1+t2+t3) + c(t2+t3) c(t1+t2)] (not symmetric in
    the delays: pins the operator order and the time arguments).  Compact scheme on the h = 0.5 mesh."""
    def c(t):
        return scipy.linalg.expm(t * bo_matrix())[0, 1]
    dt = 5e-3
    t1s, t2s, t3s = [0, 100], [60, 140], [0, 80, 180]
    mu, al = ci.observable("mu", 1), ci.observable("alpha", 1)
    cfg = dict(harmonic(37, kp=6, depth=4), scheme="compact6")
    res = {}
    for name, ops in (("a", (mu, al, al, mu)), ("b", (mu, mu, al, al))):
        o = hermite.RefHermite(cfg)
        o.equilibrate()
        res[name] = o.response_3d(*ops, t1s, t2s, t3s, dt)
    worst = 0.0
    for k, a in enumerate(t1s):
        for j, b in enumerate(t2s):
            for l, d in enumerate(t3s):
                a_, b_, d_ = a * dt, b * dt, d * dt
                worst = max(worst, abs(res["a"][k, j, l] + 4 * c(a_) * c(b_) * c(d_)),
                            abs(res["b"][k, j, l] + 4 * c(d_) * (c(b_) * c(a_ + b_ + d_) + c(b_ + d_) * c(a_ + b_))))
    assert worst < 3e-4, worst                                   # 1e-4 of the largest value (3.2) on the h = 0.5 mesh
    assert abs(res["a"][1, 1, 2]) > 0.8 and abs(res["b"][1, 1, 2]) > 3.0

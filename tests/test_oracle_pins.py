"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only, `-m "not gpu"`).

None of these tests re-types an oracle formula: they compare it with closed forms (Brownian-oscillator
response, exact moment ODEs), invariants (Boltzmann stationarity order, norm contraction, conservation),
textbook limits (rigid rotation), convergence orders, and an independent sparse Kronecker assembly of
Eq. (8) written here with numpy/scipy.  Citations: PAPER.md line numbers; pins P1-P10 of DESIGN.md.
"""
import math
import os

import numpy as np
import pytest
import scipy.linalg
import scipy.sparse as sp

import chfpe_inputs as ci
import oracle
from conftest import make_obs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def obs(kind, M):
    return make_obs(oracle, ci.observable(kind, M))


def load_gold(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([float(x) for x in line.split()])
    return np.array(rows)


def bo_response(t, w0=1.0, zeta=0.5, gamma=1.0, m=1.0):
    """R_phys(t) = (1/m) sum_i (s_i + gamma)/D'(s_i) exp(s_i t), D(s) = s^3 + g s^2 + (w0^2 + zeta g) s + g w0^2."""
    r = np.roots([1.0, gamma, w0 * w0 + zeta * gamma, gamma * w0 * w0])
    dp = 3 * r * r + 2 * gamma * r + (w0 * w0 + zeta * gamma)
    t = np.asarray(t, dtype=float)
    return np.real(sum((ri + gamma) / di * np.exp(ri * t) for ri, di in zip(r, dp))) / m


def harmonic_cfg(n=64, half=6.0, depth=8, gauge="w", scheme="central4", w0=1.0, zeta=0.5, gamma=1.0, vsl=0.0):
    return dict(n_modes=1, U=[(0.5 * w0 * w0, (2,))], V_LL=[1.0], V_SL=[vsl], zeta=[zeta], gamma=[gamma],
                beta=1.0, mass=[1.0], depth=depth, nq=[n], np=[n], qmin=[-half], qmax=[half], pmin=[-half],
                pmax=[half], scheme=scheme, gauge=gauge)


# ----------------------------------------------------------------------------- structure
def test_element_sets_and_order():
    """R5/R6: simplex sum n_s <= N, graded then descending-lex; BASELINE counts 9 / 15 / 20."""
    o = oracle.RefCHFPE(ci.config("cfg3s", depth=2, nq=[5, 5], np=[5, 5]))
    assert o.elements() == [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]
    assert oracle.RefCHFPE(ci.config("cfg1")).K == 9
    assert oracle.RefCHFPE(ci.config("cfg3s", nq=[5, 5], np=[5, 5])).K == 15
    o3 = oracle.RefCHFPE(ci.config("cfg4s8", nq=[5] * 3, np=[5] * 3))
    assert o3.K == 20
    el = o3.elements()
    assert len(set(el)) == 20 and all(sum(n) <= 3 for n in el)
    for k, n in enumerate(el):
        for s in range(3):
            up, dn = o3.neighbor(k, s)
            nu = list(n); nu[s] += 1
            nd = list(n); nd[s] -= 1
            assert (up == -1) == (sum(nu) > 3) and (up < 0 or el[up] == tuple(nu))
            assert (dn == -1) == (nd[s] < 0) and (dn < 0 or el[dn] == tuple(nd))


# ----------------------------------------------------------------------------- P1
@pytest.mark.parametrize("gauge,tol", [("w", 5e-8), ("sqrt_eq", 6e-5)])
def test_P1_brownian_oscillator_closed_form(gauge, tol):
    """Config 1: literal Eq. (15) = -R_phys of the closed form (reading R3)."""
    cfg = ci.config("cfg1", gauge=gauge)
    o = oracle.RefCHFPE(cfg)
    o.equilibrate()
    assert abs(o.expect(obs("one", 1)) - 1.0) < 1e-13
    R = o.response_1d(obs("mu", 1), obs("mu", 1), 2001, 1, cfg["dt"])
    t = np.arange(2001) * cfg["dt"]
    assert np.max(np.abs(-R - bo_response(t))) < tol
    gold = load_gold("bo_response_cfg1.txt")
    for tt, val in gold:
        assert abs(bo_response(tt) - val) < 1e-9          # the fixture is the closed form
        assert abs(-R[int(round(tt / cfg["dt"]))] - val) < tol


def test_P1_compact6_sqrt_gauge():
    """COMPACT6 with a = 7/9 (reading R4) reaches 5e-8-level agreement in the sqrt(W_eq) gauge."""
    cfg = ci.config("cfg1", scheme="compact6")
    o = oracle.RefCHFPE(cfg)
    o.equilibrate()
    R = o.response_1d(obs("mu", 1), obs("mu", 1), 11, 100, 1e-3)
    assert np.max(np.abs(-R - bo_response(np.arange(11) * 0.1))) < 2e-7


# ----------------------------------------------------------------------------- SL coupling (V'_s of PAPER.md:65)
def _short_time_t2_coefficient(R_lib, dt):
    """Least-squares fit of R_phys(t)/t = c0 + c2 t^2 + c3 t^3 + c4 t^4 + c5 t^5 on the sampled window; returns (c0, c2)."""
    t = np.arange(1, len(R_lib)) * dt
    f = -np.asarray(R_lib)[1:] / t
    A = np.stack([t ** k for k in (0, 2, 3, 4, 5)], axis=1)
    c = np.linalg.lstsq(A, f, rcond=None)[0]
    return c[0], c[1]


@pytest.mark.parametrize("which", ["grid_w_gauge", "hermite"])
def test_short_time_expansion_pins_Vprime(which):
    """V'_s(q) = V_LL + V_SL q (Eq. 11-12 :96-100) pinned by mathematics, not by a copy of itself.

    Generalised Langevin picture behind Eq. (8): q'' = (-U' + V'(q) Omega)/m,
    Omega' = -gamma Omega - zeta gamma V'(q) p + noise, R_phys(t) = <dq(t)/dp(0)>_eq.  Expanding in t:
        R_phys(t) = t/m - [ <U''>/m + zeta gamma <V'(q)^2>_eq ] t^3 / (6 m) + O(t^4),
    and for harmonic U:  <V'^2>_eq = V_LL^2 + V_SL^2 / (beta m w0^2)  (the cross term is odd in q).
    V_SL = 0 must reproduce the closed form's -(w0^2 + zeta gamma)/6; a slip such as V_SL q / 2 gives
    -0.2708 instead of -0.3333 at V_SL = 1 and fails (tried: editing Vprime / self.Vp that way fails this test).
    """
    from oracle import hermite
    w0, zeta, gamma, beta, m, vll = 1.0, 0.5, 1.0, 1.0, 1.0, 1.0
    mu = ci.observable("mu", 1)
    for vsl in (0.0, 1.0):
        cfg = dict(n_modes=1, U=[(0.5 * m * w0 * w0, (2,))], V_LL=[vll], V_SL=[vsl], zeta=[zeta], gamma=[gamma],
                   beta=beta, mass=[m], depth=4, nq=[96], np=[96], qmin=[-8.0], qmax=[8.0], pmin=[-8.0], pmax=[8.0],
                   scheme="central4", gauge="w")
        if which == "hermite":
            cfg.update(np=[12], gauge="sqrt_eq")
            o = hermite.RefHermite(cfg)
            o.equilibrate()
            R = o.response_1d(mu, mu, 201, 1, 1e-3)
        else:
            o = oracle.RefCHFPE(cfg)
            o.equilibrate()
            R = o.response_1d(obs("mu", 1), obs("mu", 1), 201, 1, 1e-3)
        c0, c2 = _short_time_t2_coefficient(R, 1e-3)
        expect = -(w0 ** 2 + zeta * gamma * (vll ** 2 + vsl ** 2 / (beta * m * w0 ** 2))) / (6.0 * m)
        assert abs(c0 - 1.0 / m) < 5e-5
        assert abs(c2 - expect) < 1e-3 * abs(expect), (which, vsl, c2, expect)
    assert abs(expect - (-1.0 / 3.0)) < 1e-12 and abs(-(w0 ** 2 + zeta * gamma) / 6.0 - (-0.25)) < 1e-12


# ----------------------------------------------------------------------------- terminator closure (reading R23)
@pytest.mark.parametrize("gauge,tol", [("w", 1e-7), ("sqrt_eq", 8e-5)])
def test_terminator_depth0_is_the_kramers_equation(gauge, tol):
    """Depth 0 with the terminator: W^(e_s) = Theta_s W^(0) / gamma_s turns Phi_s W^(e_s) into the Fokker-Planck term
    zeta_s V'_s^2 d/dp (p + (m/beta) d/dp): the Markovian Kramers equation with friction zeta V'^2, independent of
    gamma.  Harmonic U, V' = 1: the damped oscillator s^2 + zeta s + w0^2, R_phys(t) = exp(-zeta t/2) sin(Omega t)/(m Omega)."""
    w0, zeta = 1.0, 0.5
    t = np.arange(21) * 0.1
    Om = math.sqrt(w0 * w0 - zeta * zeta / 4.0)
    exact = np.exp(-zeta * t / 2.0) * np.sin(Om * t) / Om
    for gamma in (1.0, 3.0):
        cfg = harmonic_cfg(depth=0, gauge=gauge, zeta=zeta, gamma=gamma)
        cfg["closure"] = "terminator"
        o = oracle.RefCHFPE(cfg)
        o.equilibrate()
        R = o.response_1d(obs("mu", 1), obs("mu", 1), 21, 100, 1e-3)
        assert np.max(np.abs(-R - exact)) < tol, (gauge, gamma)
    cfg["closure"] = "truncate"                                  # plain truncation at depth 0 has no bath at all
    o = oracle.RefCHFPE(cfg)
    o.equilibrate()
    R = o.response_1d(obs("mu", 1), obs("mu", 1), 21, 100, 1e-3)
    assert np.max(np.abs(-R - np.sin(w0 * t) / w0)) < 1e-4 and np.max(np.abs(-R - exact)) > 0.1


def test_terminator_needs_fewer_levels():
    """Anharmonic mode with LL+SL coupling and a fast bath (config 2 with gamma = 6): at every depth 0..3 the terminator
    is closer to the converged hierarchy (depth 10) than plain truncation, and it reaches 1e-4 one level earlier."""
    def resp(depth, closure):
        cfg = ci.config("cfg2", depth=depth, nq=[64], np=[64], gamma=[6.0], closure=closure)
        o = oracle.RefCHFPE(cfg)
        o.equilibrate()
        return o.response_1d(obs("mu_nl", 1), obs("mu_nl", 1), 41, 100, cfg["dt"])
    ref = resp(10, "truncate")
    assert np.max(np.abs(resp(10, "terminator") - ref)) < 1e-10   # both closures converge to the same hierarchy
    err = {c: [float(np.max(np.abs(resp(N, c) - ref))) for N in range(4)] for c in ("truncate", "terminator")}
    for N in range(4):
        assert err["terminator"][N] < 0.5 * err["truncate"][N], (N, err)
    first = {c: next(N for N in range(4) if err[c][N] < 1e-4) for c in err}
    assert first["terminator"] < first["truncate"], (first, err)


# ----------------------------------------------------------------------------- P3
def test_P3_second_moment_ode_pins_down_coupling_factor():
    """Exact 6x6 second-moment ODE (harmonic + LL); wrong by 3e-2 without the n_s of reading R1."""
    m = w0 = beta = 1.0
    zeta, gamma = 0.5, 1.0
    # y = (<q2>, <qp>, <p2>, <qO>, <pO>, <O2>), kicked part has <1> = 0
    A = np.array([[0, 2 / m, 0, 0, 0, 0],
                  [-m * w0 ** 2, 0, 1 / m, 1, 0, 0],
                  [0, -2 * m * w0 ** 2, 0, 0, 2, 0],
                  [0, -zeta * gamma, 0, -gamma, 1 / m, 0],
                  [0, 0, -zeta * gamma, -m * w0 ** 2, -gamma, 1],
                  [0, 0, 0, 0, -2 * zeta * gamma, -2 * gamma]], dtype=float)
    y0 = np.array([0, -2 / (beta * m * w0 ** 2), 0, 0, 0, 0], dtype=float)
    y2 = scipy.linalg.expm(2.0 * A) @ y0
    gold = load_gold("moment_q2_cfg1.txt")
    assert abs(y2[0] - gold[0, 1]) < 1e-9
    sigma2 = m * zeta * gamma / beta
    for depth in (2, 8):
        o = oracle.RefCHFPE(harmonic_cfg(depth=depth))
        o.equilibrate()
        o.kick(obs("alpha", 1))
        o.step(2000, 1e-3)
        q2 = oracle.make_observable(quad=[[2.0]])
        assert abs(o.expect(q2) - y2[0]) < 1e-6
        # <q Omega> = - int q W^(1),  <Omega^2> = sigma^2 int W^(0) + int W^(2)
        qO = -o.expect(oracle.make_observable(lin_q=[1.0]), element=1)
        O2 = sigma2 * o.expect(obs("one", 1)) + o.expect(obs("one", 1), element=2)
        pO = -o.expect(oracle.make_observable(lin_p=[1.0]), element=1)
        assert abs(qO - y2[3]) < 1e-6 and abs(pO - y2[4]) < 1e-6 and abs(O2 - y2[5]) < 1e-6
    o1 = oracle.RefCHFPE(harmonic_cfg(depth=1))      # depth 1 cannot close the second moments
    o1.equilibrate(); o1.kick(obs("alpha", 1)); o1.step(2000, 1e-3)
    assert abs(o1.expect(oracle.make_observable(quad=[[2.0]])) - y2[0]) > 1e-2


def test_P3_first_moment_ode():
    """<q>,<p>,<Omega> obey the 3x3 linear ODE; <Omega> = - int W^(1)."""
    zeta, gamma = 0.5, 1.0
    A = np.array([[0, 1, 0], [-1, 0, 1], [0, -zeta * gamma, -gamma]], dtype=float)
    y = scipy.linalg.expm(1.5 * A) @ np.array([0.0, -1.0, 0.0])
    o = oracle.RefCHFPE(harmonic_cfg(depth=3))
    o.equilibrate(); o.kick(obs("mu", 1)); o.step(1500, 1e-3)
    got = [o.expect(oracle.make_observable(lin_q=[1.0])), o.expect(oracle.make_observable(lin_p=[1.0])),
           -o.expect(obs("one", 1), element=1)]
    assert np.max(np.abs(np.array(got) - y)) < 5e-8


# ----------------------------------------------------------------------------- P2
def test_P2_boltzmann_stationarity_order4():
    """Anharmonic U with LL+SL coupling: ||F(X_eq)|| -> 0 as h^4 at level 0 (signs of L) and level 1 (Theta)."""
    r0, r1 = [], []
    for n in (32, 64, 128):
        cfg = ci.config("cfg2", gauge="w", depth=3, nq=[n], np=[n])
        o = oracle.RefCHFPE(cfg)
        o.equilibrate()
        X = o.export_state()
        F = o.rhs(X)
        nx = np.linalg.norm(X)
        r0.append(np.linalg.norm(F[0]) / nx)
        r1.append(np.linalg.norm(F[1]) / nx)
        assert np.linalg.norm(F[2:]) == 0.0
    for r in (r0, r1):
        assert 12.0 < r[0] / r[1] < 20.0 and 14.0 < r[1] / r[2] < 18.0
    assert r0[2] < 1e-4 and r1[2] < 2e-4


def test_P2_stationarity_sqrt_gauge_two_modes():
    """Same invariant through the sqrt(W_eq) gauge, two coupled modes (cross term + SL)."""
    res = []
    for n in (12, 24):
        cfg = ci.config("cfg3s", depth=2, nq=[n, n], np=[n, n])
        res.append(oracle.RefCHFPE(cfg).equilibrate())
    assert res[0] / res[1] > 10.0


# ----------------------------------------------------------------------------- P4
def test_P4_two_dimensional_closed_form():
    """R2_lib(t2,t1) = 2 R_phys(t1) R_phys(t2) for A=C=q, B=q^2 (harmonic + LL); zero when B is linear."""
    gold = load_gold("r2_closed_form.txt")[0]
    assert abs(2 * bo_response(gold[0]) * bo_response(gold[1]) - gold[2]) < 1e-8
    o = oracle.RefCHFPE(harmonic_cfg(n=48, depth=4))
    o.equilibrate()
    R = o.response_2d(obs("mu", 1), obs("alpha", 1), obs("mu", 1), [0, 800], [0, 1200], 1e-3)
    assert abs(R[1, 1] - gold[2]) < 1e-6
    assert abs(R[0, 1] - 2 * bo_response(0.0) * bo_response(1.2)) < 1e-6
    o.equilibrate()
    R0 = o.response_2d(obs("mu", 1), obs("mu", 1), obs("mu", 1), [800], [1200], 1e-3)
    assert abs(R0[0, 0]) < 1e-7


def test_P4b_third_order_closed_forms():
    """Eq. (17) PAPER.md:126-127 on the harmonic + LL model, where E[q(t) | q0, p0, Omega0] is linear with
    d E[q(t)] / d p0 = R_phys(t) =: c(t): integrating each kick by parts (int f X^x W = -int (dX/dq)(df/dp) W) gives
      A = D = q, B = C = q^2:   R3_lib = -4 c(t1) c(t2) c(t3)
      A = B = q, C = D = q^2:   R3_lib = -4 c(t3) [ c(t2) c(t1+t2+t3) + c(t2+t3) c(t1+t2) ]
    (the second is not symmetric in the delays: it pins the order of the operators and of the time arguments), and
    zero if fewer than two of the four operators are quadratic."""
    c = bo_response
    dt = 1e-3
    t1s, t2s, t3s = [0, 500], [300, 700], [0, 400, 900]
    mu, al = obs("mu", 1), obs("alpha", 1)
    o = oracle.RefCHFPE(harmonic_cfg(n=48, depth=4))
    o.equilibrate()
    Ra = o.response_3d(mu, al, al, mu, t1s, t2s, t3s, dt)
    o.equilibrate()
    Rb = o.response_3d(mu, mu, al, al, t1s, t2s, t3s, dt)
    o.equilibrate()
    Rz = o.response_3d(mu, mu, al, mu, t1s, t2s, t3s, dt)
    for k, a in enumerate(t1s):
        for j, b in enumerate(t2s):
            for l, d in enumerate(t3s):
                a_, b_, d_ = a * dt, b * dt, d * dt
                assert abs(Ra[k, j, l] + 4 * c(a_) * c(b_) * c(d_)) < 3e-5
                assert abs(Rb[k, j, l] + 4 * c(d_) * (c(b_) * c(a_ + b_ + d_) + c(b_ + d_) * c(a_ + b_))) < 3e-5
                assert abs(Rz[k, j, l]) < 3e-5
    assert abs(Ra[1, 1, 2]) > 0.8 and abs(Rb[1, 1, 2]) > 3.0     # the tolerances above are 1e-5 relative


def test_response_3d_equals_manual_protocol():
    """Eq. (17) order of operations: kick A, t1, kick B, t2, kick C, t3, <D>."""
    cfg = ci.config("cfg2", nq=[24], np=[24], depth=3)
    o = oracle.RefCHFPE(cfg)
    o.equilibrate()
    t1s, t2s, t3s = [0, 3], [1, 4], [0, 2, 5]
    R = o.response_3d(obs("mu", 1), obs("alpha", 1), obs("mu_nl", 1), obs("alpha", 1), t1s, t2s, t3s, 1e-2)
    for k, a in enumerate(t1s):
        for j, b in enumerate(t2s):
            for l, d in enumerate(t3s):
                o.equilibrate(); o.kick(obs("mu", 1)); o.step(a, 1e-2); o.kick(obs("alpha", 1)); o.step(b, 1e-2)
                o.kick(obs("mu_nl", 1)); o.step(d, 1e-2)
                assert abs(o.expect(obs("alpha", 1)) - R[k, j, l]) <= 1e-14 * max(1.0, abs(R[k, j, l]))


def test_response_2d_equals_manual_protocol():
    """Eq. (16) order of operations: kick A, t1, kick B, t2, <C>."""
    cfg = ci.config("cfg2", nq=[24], np=[24], depth=3)
    o = oracle.RefCHFPE(cfg)
    o.equilibrate()
    R = o.response_2d(obs("mu", 1), obs("alpha", 1), obs("mu_nl", 1), [0, 3, 7], [0, 2, 5], 1e-2)
    for k, a in enumerate([0, 3, 7]):
        for j, b in enumerate([0, 2, 5]):
            o.equilibrate(); o.kick(obs("mu", 1)); o.step(a, 1e-2); o.kick(obs("alpha", 1)); o.step(b, 1e-2)
            assert abs(o.expect(obs("mu_nl", 1)) - R[k, j]) <= 1e-14 * max(1.0, abs(R[k, j]))


# ----------------------------------------------------------------------------- P5
def test_P5_rigid_rotation_limit():
    """zeta = 0: R_phys = sin(w0 t)/(m w0); the hierarchy decouples."""
    w0 = 1.3
    o = oracle.RefCHFPE(harmonic_cfg(depth=2, zeta=0.0, w0=w0))
    o.equilibrate()
    R = o.response_1d(obs("mu", 1), obs("mu", 1), 5, 250, 2e-3)
    t = np.arange(5) * 0.5
    assert np.max(np.abs(-R - np.sin(w0 * t) / w0)) < 2e-7


def test_P5_markov_limit_is_damped_oscillator():
    """gamma -> infinity at fixed zeta: s^2 + zeta s + w0^2 (Kramers friction); reading R21."""
    zeta, gamma = 0.4, 200.0
    o = oracle.RefCHFPE(harmonic_cfg(n=48, depth=3, zeta=zeta, gamma=gamma))
    o.equilibrate()
    R = o.response_1d(obs("mu", 1), obs("mu", 1), 4, 250, 2e-3)
    t = np.arange(4) * 0.5
    wd = math.sqrt(1.0 - zeta * zeta / 4)
    kram = np.exp(-zeta * t / 2) * np.sin(wd * t) / wd
    assert np.max(np.abs(-R - kram)) < 5e-3                # O(1/gamma) correction
    assert np.max(np.abs(-R - bo_response(t, zeta=zeta, gamma=gamma))) < 1e-6


# ----------------------------------------------------------------------------- P6, P7
def test_P6_scaled_norm_contraction_sqrt_gauge():
    """sum_n ||X_n||^2 / prod n_s!(zeta gamma m/beta)^n_s is non-increasing for any U, V, M (central schemes)."""
    cfg = ci.config("cfg3s", depth=2, nq=[10, 9], np=[11, 10])
    o = oracle.RefCHFPE(cfg)
    X = ci.seeded_state(cfg, [sum(n) for n in o.elements()], seed=3)
    o.import_state(X)
    norms = [o.scaled_norm2()]
    for _ in range(6):
        o.step(25, 1e-2)
        norms.append(o.scaled_norm2())
    assert all(b <= a * (1 + 1e-12) for a, b in zip(norms, norms[1:]))
    assert norms[-1] < 0.95 * norms[0]


def test_P6_generator_is_skew_plus_damping():
    """Assembled sqrt-gauge operator (from oracle RHS columns): symmetric part of the scaled generator = -Gamma."""
    cfg = harmonic_cfg(n=8, depth=2, gauge="sqrt_eq", vsl=0.3)
    cfg["np"] = [9]
    cfg["U"] = [(0.5, (2,)), (-0.05, (3,)), (0.01, (4,))]
    o = oracle.RefCHFPE(cfg)
    N = o.K * o.cells
    L = np.empty((N, N))
    for j in range(N):
        e = np.zeros(N); e[j] = 1.0
        L[:, j] = o.rhs(e).reshape(-1)
    cdn = cfg["zeta"][0] * cfg["gamma"][0]
    scale = np.repeat([math.sqrt(math.factorial(n) * cdn ** n) for n in range(o.K)], o.cells)
    Ls = L * scale[None, :] / scale[:, None]
    S = 0.5 * (Ls + Ls.T)
    expect = -np.repeat([n * cfg["gamma"][0] for n in range(o.K)], o.cells)
    assert np.max(np.abs(S - np.diag(expect))) < 1e-12


def test_P7_conservation_of_W0_in_W_gauge():
    """d/dt int W^(0) = 0 up to the boundary tail mass; literal Eq. (8)."""
    cfg = harmonic_cfg(n=48, half=8.0, depth=3, vsl=0.2)
    o = oracle.RefCHFPE(cfg)
    q = np.linspace(-8, 8, 48)
    X = np.zeros((o.K, 48, 48))
    X[0] = np.exp(-((q[:, None] - 1.0) ** 2) - (q[None, :] + 0.5) ** 2)
    X[1] = 0.3 * np.exp(-(q[:, None] ** 2) - (q[None, :] - 0.7) ** 2)
    o.import_state(X)
    one = obs("one", 1)
    n0 = o.expect(one)
    o.step(300, 2e-3)
    assert abs(o.expect(one) - n0) < 1e-10 * abs(n0)


# ----------------------------------------------------------------------------- P8
def test_P8_additivity_uncoupled_modes():
    """Uncoupled harmonic modes, mu = q1 + q2: R1 = R1_mode1 + R1_mode2 -- against the closed forms and against
    two one-mode runs on the same per-axis grids (tail-mass limited; W gauge; distinct sizes per axis)."""
    w = (1.0, 1.3); zeta = (0.5, 0.8); gamma = (1.0, 0.7); n = 16; half = 5.0
    base = dict(beta=1.0, depth=2, scheme="central4", gauge="w")
    cfg = dict(base, n_modes=2, U=[(0.5 * w[0] ** 2, (2, 0)), (0.5 * w[1] ** 2, (0, 2))], V_LL=[1.0, 1.0],
               V_SL=[0.0, 0.0], zeta=list(zeta), gamma=list(gamma), mass=[1.0, 1.0], nq=[n, n + 1], np=[n + 2, n],
               qmin=[-half] * 2, qmax=[half] * 2, pmin=[-half] * 2, pmax=[half] * 2)
    o = oracle.RefCHFPE(cfg)
    o.equilibrate()
    R = o.response_1d(obs("mu", 2), obs("mu", 2), 3, 50, 5e-3)
    t = np.arange(3) * 0.25
    exact = sum(bo_response(t, w0=w[s], zeta=zeta[s], gamma=gamma[s]) for s in range(2))
    assert np.max(np.abs(-R - exact)) < 6e-5
    Rs = 0.0
    for s in range(2):
        c1 = dict(base, n_modes=1, U=[(0.5 * w[s] ** 2, (2,))], V_LL=[1.0], V_SL=[0.0], zeta=[zeta[s]],
                  gamma=[gamma[s]], mass=[1.0], nq=[cfg["nq"][s]], np=[cfg["np"][s]], qmin=[-half], qmax=[half],
                  pmin=[-half], pmax=[half])
        o1 = oracle.RefCHFPE(c1)
        o1.equilibrate()
        Rs = Rs + o1.response_1d(obs("mu", 1), obs("mu", 1), 3, 50, 5e-3)
    assert np.max(np.abs(R - Rs)) < 3e-6


# ----------------------------------------------------------------------------- P9
def test_P9_rk4_order_in_dt():
    cfg = ci.config("cfg2", nq=[32], np=[32], depth=4)
    vals = []
    for nst, dt in ((20, 0.02), (40, 0.01), (160, 0.0025)):
        o = oracle.RefCHFPE(cfg)
        o.equilibrate(); o.kick(obs("mu_nl", 1)); o.step(nst, dt)
        vals.append(o.export_state())
    e1 = np.linalg.norm(vals[0] - vals[2]); e2 = np.linalg.norm(vals[1] - vals[2])
    assert 13.0 < e1 / e2 < 19.0


def test_P9_depth_convergence_anharmonic_sl():
    cfg0 = ci.config("cfg2", nq=[40], np=[40])
    vals = []
    for depth in (3, 6, 9, 12):
        o = oracle.RefCHFPE(dict(cfg0, depth=depth))
        o.equilibrate()
        vals.append(o.response_1d(obs("mu_nl", 1), obs("mu_nl", 1), 5, 100, 5e-3))
    d = [np.max(np.abs(a - b)) for a, b in zip(vals, vals[1:])]
    assert d[0] > d[1] > d[2] and d[2] < 1e-6


def test_compact6_is_sixth_order_with_corrected_constants():
    """Reading R4: a = 7/9, b = 1/36, alpha = 1/3 gives order 6 (7/18 is not even consistent)."""
    errs = []
    for n in (33, 65):
        cfg = harmonic_cfg(n=n, half=8.0, depth=0, scheme="compact6")
        o = oracle.RefCHFPE(cfg)
        x = np.linspace(-8, 8, n)
        f = np.exp(-0.5 * x[:, None] ** 2) * np.exp(-0.25 * x[None, :] ** 2)
        dq = o.deriv_axis(f, 0)
        dp = o.deriv_axis(f, 1)
        errs.append(max(np.max(np.abs(dq + x[:, None] * f)), np.max(np.abs(dp + 0.5 * x[None, :] * f))))
    assert 45.0 < errs[0] / errs[1] < 100.0 and errs[1] < 1e-5


def test_central_orders():
    for scheme, lo, hi in (("central4", 13.0, 18.0), ("central2", 3.6, 4.4)):
        errs = []
        for n in (65, 129):
            o = oracle.RefCHFPE(harmonic_cfg(n=n, half=8.0, depth=0, scheme=scheme))
            x = np.linspace(-8, 8, n)
            f = np.exp(-0.5 * x[:, None] ** 2) * np.exp(-0.25 * x[None, :] ** 2)
            errs.append(np.max(np.abs(o.deriv_axis(f, 0) + x[:, None] * f)))
        assert lo < errs[0] / errs[1] < hi


# ----------------------------------------------------------------------------- P10: independent assembly
def _d_matrix(n, h, scheme):
    """Dense 1-D derivative matrix with zero ghosts: explicit stencils or A^-1 B of Eq. (28)-(29)."""
    def band(k):
        return np.eye(n, k=k) - np.eye(n, k=-k)
    if scheme == "central4":
        return (8 * band(1) - band(2)) / (12 * h)
    if scheme == "central2":
        return band(1) / (2 * h)
    A = np.eye(n) + (np.eye(n, k=1) + np.eye(n, k=-1)) / 3.0
    B = (7.0 / 9.0 * band(1) + 1.0 / 36.0 * band(2)) / h
    return np.linalg.solve(A, B)


def _assemble(cfg, elements):
    """Sparse generator of Eq. (8) on the canonical layout, built from Kronecker products (numpy/scipy only)."""
    M = cfg["n_modes"]
    sizes, coords = [], []
    for s in range(M):
        sizes += [cfg["nq"][s], cfg["np"][s]]
        coords += [np.linspace(cfg["qmin"][s], cfg["qmax"][s], cfg["nq"][s]),
                   np.linspace(cfg["pmin"][s], cfg["pmax"][s], cfg["np"][s])]
    cells = int(np.prod(sizes))

    def kron_axis(mat, ax):
        out = sp.identity(1, format="csr")
        for a, n in enumerate(sizes):
            out = sp.kron(out, sp.csr_matrix(mat) if a == ax else sp.identity(n, format="csr"), format="csr")
        return out

    def diag_of(fn):
        grids = np.meshgrid(*coords, indexing="ij")
        return sp.diags(fn(grids).reshape(-1))

    D = [kron_axis(_d_matrix(sizes[a], coords[a][1] - coords[a][0], cfg["scheme"]), a) for a in range(2 * M)]

    def dU(s):
        def fn(g):
            out = np.zeros_like(g[0])
            for coef, expo in cfg["U"]:
                if expo[s] == 0:
                    continue
                term = coef * expo[s] * g[2 * s] ** (expo[s] - 1)
                for r in range(M):
                    if r != s:
                        term = term * g[2 * r] ** expo[r]
                out = out + term
            return out
        return diag_of(fn)

    beta = cfg["beta"]
    K = len(elements)
    index = {n: k for k, n in enumerate(elements)}
    blocks = [[None] * K for _ in range(K)]
    for k, n in enumerate(elements):
        Lk = -sum(n[s] * cfg["gamma"][s] for s in range(M)) * sp.identity(cells, format="csr")
        for s in range(M):
            m = cfg["mass"][s]
            P = diag_of(lambda g: g[2 * s + 1])
            Vp = diag_of(lambda g: cfg["V_LL"][s] + cfg["V_SL"][s] * g[2 * s])
            Lk = Lk - (P / m) @ D[2 * s] + dU(s) @ D[2 * s + 1]
            if cfg["gauge"] == "w":
                kup, kdn = 0.0, beta / m
            else:
                kup, kdn = -beta / (2 * m), beta / (2 * m)
            nu = list(n); nu[s] += 1
            if tuple(nu) in index:
                blocks[k][index[tuple(nu)]] = Vp @ (D[2 * s + 1] + kup * P)
            nd = list(n); nd[s] -= 1
            if nd[s] >= 0:
                c = cfg["zeta"][s] * cfg["gamma"][s] * m / beta
                blocks[k][index[tuple(nd)]] = n[s] * c * (Vp @ (D[2 * s + 1] + kdn * P))
            if cfg.get("closure") == "terminator" and sum(n) == cfg["depth"]:
                # reading R23: W^(n+e_s) = (n_s+1) Theta_s W^(n) / Gamma_{n+e_s}, fed back through Phi_s (Eq. 11, 12)
                c = cfg["zeta"][s] * cfg["gamma"][s] * m / beta
                gam_up = sum(n[r] * cfg["gamma"][r] for r in range(M)) + cfg["gamma"][s]
                Lk = Lk + ((n[s] + 1) * c / gam_up) * (Vp @ (D[2 * s + 1] + kup * P)) @ (Vp @ (D[2 * s + 1] + kdn * P))
        blocks[k][k] = Lk
    return sp.bmat(blocks, format="csr"), D, coords


def _with(cfg, **over):
    c = dict(cfg)
    c.update(over)
    return c


ASSEMBLY_CASES = [
    ("m1_c4_w", dict(n_modes=1, U=[(0.5, (2,)), (-0.05, (3,)), (0.004, (4,))], V_LL=[0.9], V_SL=[0.3], zeta=[0.7],
                     gamma=[1.3], beta=0.8, mass=[1.7], depth=3, nq=[9], np=[11], qmin=[-3.0], qmax=[3.5],
                     pmin=[-4.0], pmax=[4.5], scheme="central4", gauge="w")),
    ("m1_c2_sqrt", dict(n_modes=1, U=[(0.5, (2,)), (0.02, (3,))], V_LL=[1.0], V_SL=[-0.2], zeta=[0.4],
                        gamma=[0.9], beta=1.2, mass=[0.6], depth=2, nq=[8], np=[7], qmin=[-3.0], qmax=[3.0],
                        pmin=[-2.5], pmax=[2.5], scheme="central2", gauge="sqrt_eq")),
    ("m1_pade_sqrt", dict(n_modes=1, U=[(0.5, (2,)), (0.01, (4,))], V_LL=[1.0], V_SL=[0.25], zeta=[1.1],
                          gamma=[2.0], beta=1.0, mass=[1.0], depth=2, nq=[10], np=[9], qmin=[-4.0], qmax=[4.0],
                          pmin=[-4.0], pmax=[4.0], scheme="compact6", gauge="sqrt_eq")),
    ("m2_c4_sqrt", dict(n_modes=2, U=[(0.5, (2, 0)), (0.18, (0, 2)), (0.002, (4, 0)), (0.0167, (2, 1)), (0.03, (1, 1))],
                        V_LL=[1.0, 0.8], V_SL=[0.3, -0.1], zeta=[0.5, 0.9], gamma=[1.0, 0.6], beta=1.1,
                        mass=[1.0, 1.5], depth=2, nq=[6, 5], np=[7, 6], qmin=[-3.0, -4.0], qmax=[3.0, 4.5],
                        pmin=[-3.0, -2.0], pmax=[3.5, 2.0], scheme="central4", gauge="sqrt_eq")),
    ("m2_pade_w", dict(n_modes=2, U=[(0.5, (2, 0)), (0.4, (0, 2)), (0.01, (1, 2))],
                       V_LL=[1.0, 1.0], V_SL=[0.2, 0.1], zeta=[0.3, 0.4], gamma=[1.0, 2.0], beta=1.0,
                       mass=[1.0, 0.8], depth=2, nq=[5, 6], np=[6, 5], qmin=[-3.0, -3.0], qmax=[3.0, 3.0],
                       pmin=[-3.0, -3.0], pmax=[3.0, 3.0], scheme="compact6", gauge="w")),
    ("m3_c4_sqrt", dict(n_modes=3, U=[(0.5, (2, 0, 0)), (0.125, (0, 2, 0)), (0.03, (0, 0, 2)), (0.001, (0, 4, 0)),
                                      (0.008, (1, 2, 0)), (0.009, (0, 1, 2)), (0.007, (2, 0, 1)), (0.02, (1, 0, 1))],
                        V_LL=[1.0, 0.9, 1.1], V_SL=[0.2, 0.1, -0.15], zeta=[1.0, 0.65, 0.3], gamma=[0.5, 1.0, 2.0],
                        beta=0.9, mass=[1.0, 1.2, 0.7], depth=2, nq=[5, 6, 5], np=[6, 5, 7], qmin=[-3.0, -2.0, -4.0],
                        qmax=[3.0, 2.5, 4.0], pmin=[-3.0, -3.5, -2.0], pmax=[3.0, 3.0, 2.5],
                        scheme="central4", gauge="sqrt_eq")),
]
# the same operators with the terminator closure (reading R23), all three schemes, both gauges, M = 1..3
ASSEMBLY_CASES += [(nm + "_terminator", _with(c, closure="terminator")) for nm, c in
                   [ASSEMBLY_CASES[0], ASSEMBLY_CASES[1], ASSEMBLY_CASES[2], ASSEMBLY_CASES[3], ASSEMBLY_CASES[5]]]


@pytest.mark.parametrize("name,cfg", ASSEMBLY_CASES, ids=[c[0] for c in ASSEMBLY_CASES])
def test_P10_independent_kronecker_assembly(name, cfg):
    """Oracle loops == sparse Kronecker assembly of Eq. (8)-(12), (18), (15) on asymmetric tiny grids."""
    o = oracle.RefCHFPE(cfg)
    el = o.elements()
    L, D, coords = _assemble(cfg, el)
    rng = np.random.default_rng(11)
    X = rng.standard_normal((o.K,) + o.shape)
    want = (L @ X.reshape(-1)).reshape(X.shape)
    scale = np.max(np.abs(want))
    assert np.max(np.abs(o.rhs(X) - want)) < 1e-12 * scale
    assert np.max(np.abs(o.rhs(X, via_deriv=True) - want)) < 1e-12 * scale
    if cfg["scheme"] != "compact6" and cfg.get("closure", "truncate") == "truncate":
        for k, cell in ((0, 0), (o.K - 1, o.cells - 1), (1, o.cells // 3)):
            assert abs(o.rhs_at(X, k, cell) - want.reshape(o.K, -1)[k, cell]) < 1e-12 * scale
    # propagation: many small RK4 steps vs expm action
    o.import_state(X)
    o.step(200, 5e-4)
    ref = sp.linalg.expm_multiply(L * 0.1, X.reshape(-1)).reshape(X.shape)
    assert np.max(np.abs(o.export_state() - ref)) < 1e-9 * np.max(np.abs(ref))
    # kick (Eq. 18) and expectation (Eq. 15) from broadcasting
    M = cfg["n_modes"]
    lin = [0.7, -0.4, 0.3][:M]
    quad = [[0.5, 0.2, -0.1], [0.1, -0.3, 0.25], [0.05, 0.15, 0.4]]
    quad = [row[:M] for row in quad[:M]]
    ob = oracle.make_observable(c0=0.2, lin_q=lin, quad=quad, lin_p=[0.3, -0.2, 0.1][:M])
    grids = np.meshgrid(*coords, indexing="ij")
    beta = cfg["beta"]
    Hs = sum(grids[2 * s + 1] ** 2 / (2 * cfg["mass"][s]) for s in range(M))
    for coef, expo in cfg["U"]:
        term = coef
        for s in range(M):
            term = term * grids[2 * s] ** expo[s]
        Hs = Hs + term
    o.import_state(X)
    o.kick(ob)
    kicked = np.zeros_like(X)
    for k in range(o.K):
        for s in range(M):
            dXdq = lin[s] + sum(0.5 * (quad[s][r] + quad[r][s]) * grids[2 * r] for r in range(M))
            kup = 0.0 if cfg["gauge"] == "w" else -beta / (2 * cfg["mass"][s])
            dW = (D[2 * s + 1] @ X[k].reshape(-1)).reshape(o.shape) + kup * grids[2 * s + 1] * X[k]
            kicked[k] += dXdq * dW
    assert np.max(np.abs(o.export_state() - kicked)) < 1e-12 * np.max(np.abs(kicked))
    O = 0.2 + sum(lin[s] * grids[2 * s] + [0.3, -0.2, 0.1][s] * grids[2 * s + 1] for s in range(M))
    O = O + sum(0.5 * quad[a][b] * grids[2 * a] * grids[2 * b] for a in range(M) for b in range(M))
    w = 1.0 if cfg["gauge"] == "w" else np.exp(-0.5 * beta * Hs)
    dV = np.prod([c[1] - c[0] for c in coords])
    o.import_state(X)
    want_e = dV * np.sum(O * w * X[0])
    assert abs(o.expect(ob) - want_e) < 1e-12 * max(1.0, abs(want_e))
    # analytic equilibrium
    o.equilibrate()
    Xe = o.export_state()
    if cfg["gauge"] == "w":
        e0 = np.exp(-beta * Hs); e0 /= dV * e0.sum()
    else:
        e0 = np.exp(-0.5 * beta * Hs); e0 /= dV * (e0 ** 2).sum()
    assert np.max(np.abs(Xe[0] - e0)) < 1e-13 * np.max(e0) and np.all(Xe[1:] == 0)
    assert abs(o.expect(oracle.make_observable(c0=1.0)) - 1.0) < 1e-12

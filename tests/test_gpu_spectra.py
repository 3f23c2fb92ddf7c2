"""GPU parity of the spectra kernels (row f3) against oracle/spectra.py, through the C-ABI (device pointers)."""
import numpy as np
import pytest

import chfpe_inputs as ci
import oracle
from oracle import spectra
from conftest import make_obs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def gpu_mod():
    import paper_2509_25840_b200 as P
    return P


def _omega(n, hi, seed):
    rng = np.random.default_rng(seed)
    return np.concatenate([[0.0], np.sort(rng.uniform(0.0, hi, n - 1))])


@pytest.mark.parametrize("n,nw", [(1, 3), (2, 1), (33, 7), (256, 129), (2001, 40)])
def test_spectrum_1d_parity(n, nw):
    P = gpu_mod()
    rng = np.random.default_rng(n)
    t = np.arange(n) * 0.01
    R = np.exp(-0.3 * t) * np.sin(1.7 * t) + 0.1 * rng.standard_normal(n)
    om = _omega(nw, 40.0, 3)
    got, ref = P.spectrum_1d(R, 0.01, om), spectra.spectrum_1d(R, 0.01, om)
    assert got.shape == ref.shape
    assert np.max(np.abs(got - ref)) <= 1e-12 * max(1e-300, np.max(np.abs(ref)))


@pytest.mark.parametrize("n1,n2,nw1,nw2,s1,s2", [(1, 1, 1, 1, -1, -1), (5, 33, 4, 9, -1, -1), (64, 256, 37, 65, -1, -1),
                                                   (64, 256, 33, 31, -1, 1), (37, 41, 130, 3, 1, -1)])
def test_spectrum_2d_parity(n1, n2, nw1, nw2, s1, s2):
    """Sizes span several warps per row and ragged tails (delays not a multiple of 32); the paper's 64 x 256 grid."""
    P = gpu_mod()
    rng = np.random.default_rng(n1 * 1000 + n2)
    t1, t2 = np.arange(n1) * 0.02, np.arange(n2) * 0.015
    R = np.outer(np.exp(-0.4 * t1) * np.cos(2.1 * t1), np.exp(-0.2 * t2) * np.sin(3.3 * t2)) + 0.05 * rng.standard_normal((n1, n2))
    om1, om2 = _omega(nw1, 30.0, 1), _omega(nw2, 50.0, 2)
    got = P.spectrum_2d(R, 0.02, 0.015, om1, om2, s1, s2)
    ref = spectra.spectrum_2d(R, 0.02, 0.015, om1, om2, s1, s2)
    assert got.shape == ref.shape == (nw1, nw2)
    assert np.max(np.abs(got - ref)) <= 1e-12 * max(1e-300, np.max(np.abs(ref)))


def test_spectrum_errors():
    P = gpu_mod()
    with pytest.raises(P.ChfpeError):
        P.spectrum_1d([1.0, 2.0], 0.0, [1.0])                   # dt <= 0
    with pytest.raises(P.ChfpeError):
        P.spectrum_2d(np.ones((3, 4)), 0.1, 0.1, [1.0], [2.0], sign1=2)


def test_absorption_spectrum_of_config1_end_to_end():
    """R1 from the CUDA propagation -> Eq. (19) on the CUDA spectra kernel: against the oracle chain on a short
    window (2000 oracle steps), and on the full decay (t = 80, slowest mode e^{-0.12 t}) against the closed-form
    Brownian-oscillator line shape, Im of the susceptibility of the 3 x 3 first-moment ODE of pin P3."""
    P = gpu_mod()
    cfg = ci.config("cfg1")
    d = ci.observable("mu", 1)
    g, o = P.CHFPE(cfg), oracle.RefCHFPE(cfg)
    mu_g, mu_o = make_obs(P, d), make_obs(oracle, d)
    dt, stride = cfg["dt"], 50
    om = np.linspace(0.0, 3.0, 61)
    g.equilibrate(); o.equilibrate()
    Rg = g.response_1d(mu_g, mu_g, 41, stride, dt)
    Ro = o.response_1d(mu_o, mu_o, 41, stride, dt)
    Ig = P.spectrum_1d(Rg, stride * dt, om)
    Io = spectra.spectrum_1d(Ro, stride * dt, om)
    assert np.max(np.abs(Ig - Io)) <= 1e-8 * np.max(np.abs(Io))
    g.equilibrate()
    Rg = g.response_1d(mu_g, mu_g, 1601, stride, dt)
    Ig = P.spectrum_1d(Rg, stride * dt, om)
    # R_phys(t) = [e^{At}]_{01};  int_0^inf e^{iwt} R_phys dt = [(-iw - A)^{-1}]_{01};  literal Eq. (15) is -R_phys (R3)
    A = np.array([[0, 1, 0], [-1, 0, 1], [0, -0.5, -1.0]], dtype=float)
    chi = np.array([np.linalg.inv(-1j * w * np.eye(3) - A)[0, 1] for w in om])
    exact = om * (-chi.imag)
    assert np.max(np.abs(exact)) > 4.0                          # the resonance near w = 1.14
    assert np.max(np.abs(Ig - exact)) < 1e-3 * np.max(np.abs(exact))
    g.close()


def test_absorption_spectrum_in_the_papers_scheme_end_to_end():
    """The paper's own chain (section IV.C.1) on the CUDA path: Hermite representation (Eq. 22-23) with the compact
    q-derivative (Eq. 25-31) -> R1 (Eq. 15) -> spectrum (Eq. 19) against the closed-form Brownian-oscillator line
    shape of pin P3, on a 37-point q mesh (h = 0.5) with 6 Hermite functions: the spectrum is good to 2e-4 of the
    peak (trapezoid rule over the sampled decay included), where the 64 x 64 phase-space grid needs 1e-3."""
    P = gpu_mod()
    cfg = ci.config("cfg1", nq=[37], np=[6], depth=3, qmin=[-9.0], qmax=[9.0], scheme="compact6")
    g = P.Hermite(cfg)
    mu = make_obs(P, ci.observable("mu", 1))
    dt, stride = cfg["dt"], 50
    om = np.linspace(0.0, 3.0, 61)
    g.equilibrate()
    Rg = g.response_1d(mu, mu, 1601, stride, dt)
    Ig = P.spectrum_1d(Rg, stride * dt, om)
    A = np.array([[0, 1, 0], [-1, 0, 1], [0, -0.5, -1.0]], dtype=float)
    chi = np.array([np.linalg.inv(-1j * w * np.eye(3) - A)[0, 1] for w in om])
    exact = om * (-chi.imag)
    assert np.max(np.abs(Ig - exact)) < 2e-4 * np.max(np.abs(exact))
    g.close()


def test_two_dimensional_spectrum_chain_on_the_hermite_path():
    """Section IV.C.2 end to end on the CUDA path, two coupled anharmonic modes in the paper's scheme: batched
    chfpe_hermite_response_2d (Eq. 16, TRT ordering A = mu, B = alpha, C = mu) -> chfpe_spectrum_2d (Eq. 20), against
    the same chain on the oracles (oracle/hermite.py -> oracle/spectra.py)."""
    from oracle import hermite
    P = gpu_mod()
    cfg = ci.config("cfg3s", nq=[14, 12], np=[4, 4], depth=2, scheme="compact6")
    g, o = P.Hermite(cfg, batch=4), hermite.RefHermite(cfg)
    g.equilibrate(); o.equilibrate()
    mu, al = ci.observable("mu", 2), ci.observable("alpha", 2)
    stride, dt = 4, 2e-2
    t1, t2 = [stride * i for i in range(7)], [stride * i for i in range(9)]
    Rg = g.response_2d(make_obs(P, mu), make_obs(P, al), make_obs(P, mu), t1, t2, dt)
    Ro = o.response_2d(mu, al, mu, t1, t2, dt)
    assert np.max(np.abs(Ro)) > 1e-2
    assert np.max(np.abs(Rg - Ro)) <= 1e-8 * np.max(np.abs(Ro))
    om1, om2 = _omega(6, 2.0, 1), _omega(8, 2.0, 2)
    Ig = P.spectrum_2d(Rg, stride * dt, stride * dt, om1, om2)
    Io = spectra.spectrum_2d(Ro, stride * dt, stride * dt, om1, om2)
    assert np.max(np.abs(Ig - Io)) <= 1e-8 * np.max(np.abs(Io))
    g.close()

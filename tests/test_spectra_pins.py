"""Pins of the spectra oracle (oracle/spectra.py, row f3): closed-form half-line transforms, the library FFT at its
own frequencies, separability.  CPU only."""
import numpy as np

from oracle import spectra


def test_damped_sine_closed_form_and_second_order_convergence():
    """int_0^inf e^{iwt} e^{-gt} sin(Wt) dt = W / ((g - iw)^2 + W^2); the trapezoid sum converges as dt^2."""
    g, W = 0.35, 1.7
    omega = np.array([0.0, 0.4, 1.3, 1.7, 2.9])
    exact = W / ((g - 1j * omega) ** 2 + W ** 2)
    errs = []
    for dt in (0.04, 0.02, 0.01):
        t = np.arange(int(round(80.0 / dt)) + 1) * dt            # e^{-28} at the cut
        R = np.exp(-g * t) * np.sin(W * t)
        errs.append(np.max(np.abs(spectra.half_fourier_1d(R, dt, omega, +1) - exact)))
        I = spectra.spectrum_1d(R, dt, omega)
        assert np.max(np.abs(I - omega * exact.imag)) < 2.0 * errs[-1] + 1e-12
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5 and errs[2] < 2e-5


def test_sign_convention():
    """e^{+iwt} in Eq. (19), e^{-iwt} in Eq. (20): conjugate transforms of a real signal."""
    rng = np.random.default_rng(0)
    R = rng.standard_normal(37)
    om = np.array([0.3, 1.1, 2.2])
    assert np.allclose(spectra.half_fourier_1d(R, 0.1, om, +1), np.conj(spectra.half_fourier_1d(R, 0.1, om, -1)),
                       rtol=0, atol=1e-14)
    # absorption line shape: positive at the resonance of a decaying oscillation (I = w Im F)
    t = np.arange(4001) * 0.01
    assert spectra.spectrum_1d(np.exp(-0.2 * t) * np.sin(1.5 * t), 0.01, [1.5])[0] > 0


def test_reduces_to_fft_on_the_fft_grid():
    """At w_k = 2 pi k / (n dt) the rectangle sum is numpy's FFT; the trapezoid rule differs by the end weights."""
    rng = np.random.default_rng(1)
    n, dt = 64, 0.05
    R = rng.standard_normal(n)
    k = np.arange(n // 2)
    om = 2 * np.pi * k / (n * dt)
    rect = np.conj(np.fft.fft(R))[k] * dt                        # sum_j e^{+i w t_j} R_j dt
    end = 0.5 * dt * (R[0] + R[-1] * np.exp(1j * om * (n - 1) * dt))
    assert np.max(np.abs(spectra.half_fourier_1d(R, dt, om, +1) - (rect - end))) < 1e-12
    R2 = rng.standard_normal((n, n))
    rect2 = np.fft.fft2(R2)[np.ix_(k[:5], k[:7])] * dt * dt      # e^{-i w1 t1} e^{-i w2 t2}, rectangle rule
    w = np.ones(n); w[0] = w[-1] = 0.5
    trap2 = np.fft.fft2(R2 * w[:, None] * w[None, :])[np.ix_(k[:5], k[:7])] * dt * dt
    got = spectra.spectrum_2d(R2, dt, dt, om[:5], om[:7])
    assert np.max(np.abs(got - trap2.imag)) < 1e-12 and np.max(np.abs(got - rect2.imag)) > 1e-4


def test_two_dimensional_transform_is_separable():
    """R[k][j] = f(t1_k) g(t2_j)  =>  I(w1, w2) = Im[F(w1) G(w2)], also with mixed signs (Eq. 21) and dt1 != dt2."""
    t1, t2 = np.arange(40) * 0.07, np.arange(55) * 0.05
    f, gq = np.exp(-0.3 * t1) * np.cos(1.1 * t1), np.exp(-0.5 * t2) * np.sin(2.3 * t2)
    om1, om2 = np.array([0.2, 1.1, 3.0]), np.array([0.7, 2.3])
    for s1, s2 in ((-1, -1), (-1, +1)):
        F = spectra.half_fourier_1d(f, 0.07, om1, s1)
        G = spectra.half_fourier_1d(gq, 0.05, om2, s2)
        got = spectra.spectrum_2d(np.outer(f, gq), 0.07, 0.05, om1, om2, s1, s2)
        assert np.max(np.abs(got - np.outer(F, G).imag)) < 1e-13
    # transposed operand: rows are the FIRST delay
    asym = spectra.spectrum_2d(np.outer(f, gq), 0.07, 0.05, om1, om2)
    wrong = spectra.spectrum_2d(np.outer(f, gq).T.copy(), 0.05, 0.07, om2, om1).T
    assert np.max(np.abs(asym - wrong)) < 1e-13                  # consistent transposition is the identity ...
    assert np.max(np.abs(asym - spectra.spectrum_2d(np.outer(gq[:40], f), 0.07, 0.05, om1, om2))) > 1e-3   # ... swapping is not

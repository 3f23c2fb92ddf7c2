"""CPU oracle of the spectra (row f3 of DESIGN.md) -- TEST INFRASTRUCTURE, like the rest of oracle/: only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg may import it.  Shares no code with the CUDA path.

Eq. (19)-(21) PAPER.md:138-146 are half-line Fourier integrals of the sampled response functions.  The paper does
not say how they are discretised, windowed or truncated (reading R22 of DESIGN.md): here the integral over [0, T] is
the trapezoid rule on the uniform sample grid t_k = k dt, k = 0..n-1 (weights 1/2, 1, ..., 1, 1/2), no window, no
zero padding, and the frequencies are given explicitly (no FFT grid is implied).  Every function below is that
definition written out with complex exponentials in fp64.
"""
import numpy as np


def _trapezoid_weights(n):
    w = np.ones(n)
    if n > 1:
        w[0] = w[-1] = 0.5
    return w


def half_fourier_1d(R, dt, omega, sign=+1):
    """F(w) = int_0^T dt e^{i sign w t} R(t), trapezoid rule; complex array over `omega`."""
    R = np.asarray(R, dtype=np.float64)
    omega = np.asarray(omega, dtype=np.float64)
    t = np.arange(R.size) * dt
    w = _trapezoid_weights(R.size)
    out = np.empty(omega.size, dtype=np.complex128)
    for a, om in enumerate(omega):
        out[a] = np.sum(w * np.exp(1j * sign * om * t) * R) * dt
    return out


def spectrum_1d(R, dt, omega):
    """Eq. (19) :138-139: I(w) = w Im int_0^inf dt e^{i w t} R1(t)."""
    omega = np.asarray(omega, dtype=np.float64)
    return omega * half_fourier_1d(R, dt, omega, +1).imag


def spectrum_2d(R, dt1, dt2, omega1, omega2, sign1=-1, sign2=-1):
    """Eq. (20) :141-142 (sign1 = sign2 = -1): I(w1, w2) = Im int int dt1 dt2 e^{-i w1 t1} e^{-i w2 t2} R[k][j], rows of
    R along the first delay.  Eq. (21) :145-146 at a fixed waiting time is the same double transform of
    R3[:, j, :] with sign1 = -1 (t1), sign2 = +1 (t3).  Output [len(omega1)][len(omega2)]."""
    R = np.asarray(R, dtype=np.float64)
    omega1 = np.asarray(omega1, dtype=np.float64)
    omega2 = np.asarray(omega2, dtype=np.float64)
    n1, n2 = R.shape
    t1, t2 = np.arange(n1) * dt1, np.arange(n2) * dt2
    w1, w2 = _trapezoid_weights(n1), _trapezoid_weights(n2)
    out = np.empty((omega1.size, omega2.size))
    for a, oa in enumerate(omega1):
        e1 = w1 * np.exp(1j * sign1 * oa * t1)
        for b, ob in enumerate(omega2):
            e2 = w2 * np.exp(1j * sign2 * ob * t2)
            out[a, b] = (np.sum(e1[:, None] * e2[None, :] * R) * dt1 * dt2).imag
    return out

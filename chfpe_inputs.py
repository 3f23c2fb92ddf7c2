"""Seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and bench.py.

This module holds NO arithmetic of the method: only parameter dictionaries (the five BASELINE.json
configurations with the readings R14-R17 of DESIGN.md, and shrunken variants for parity tests) and a
seeded random-state generator.  The paper measures on no public data set (its workload is its own
three-mode water model); these synthetic configurations keep that structure
(1 : 0.5 : 0.25 frequency ladder, LL+SL coupling, weak cubic cross terms, one Drude bath per mode).
"""
import numpy as np


def _poly_modes(omegas, g3=None, g4=None):
    """U = sum_s [ 1/2 w_s^2 q_s^2 + g3_s q_s^3/6 + g4_s q_s^4/24 ] as (coef, exponents) monomials."""
    M = len(omegas)
    terms = []
    for s, w in enumerate(omegas):
        e = [0] * M
        e[s] = 2
        terms.append((0.5 * w * w, tuple(e)))
        if g3 is not None and g3[s] != 0.0:
            e = [0] * M
            e[s] = 3
            terms.append((g3[s] / 6.0, tuple(e)))
        if g4 is not None and g4[s] != 0.0:
            e = [0] * M
            e[s] = 4
            terms.append((g4[s] / 24.0, tuple(e)))
    return terms


def _grid(M, n, half):
    return dict(nq=[n] * M, np=[n] * M, qmin=[-half] * M, qmax=[half] * M, pmin=[-half] * M, pmax=[half] * M)


def config(name, **over):
    """Return the parameter dict of a named configuration (BASELINE.json configs 1-5 and shrunken ones)."""
    if name == "cfg1":          # 1 harmonic mode, LL coupling; closed-form Brownian-oscillator response
        c = dict(n_modes=1, U=_poly_modes([1.0]), V_LL=[1.0], V_SL=[0.0], zeta=[0.5], gamma=[1.0], beta=1.0,
                 depth=8, dt=1e-3, steps=2000, **_grid(1, 64, 6.0))
    elif name == "cfg2":        # 1 anharmonic mode, LL+SL
        c = dict(n_modes=1, U=_poly_modes([1.0], g3=[-0.3], g4=[0.05]), V_LL=[1.0], V_SL=[0.3], zeta=[1.0],
                 gamma=[2.0], beta=1.0, depth=12, dt=5e-4, steps=10000, **_grid(1, 128, 8.0))
    elif name in ("cfg3", "cfg3s"):   # 2 coupled modes, 48^4 (cfg3s: 16^4)
        n = 48 if name == "cfg3" else 16
        U = _poly_modes([1.0, 0.6], g4=[0.05, 0.05]) + [(0.1 / 6.0, (2, 1))]
        c = dict(n_modes=2, U=U, V_LL=[1.0, 1.0], V_SL=[0.3, 0.3], zeta=[0.5, 0.5], gamma=[1.0, 1.0], beta=1.0,
                 depth=4, dt=1e-3, steps=5000, **_grid(2, n, 6.0))
    elif name in ("cfg4", "cfg5", "cfg4s8", "cfg4s10", "cfg4s12", "cfg4h"):   # 3 intermolecular-like modes
        n = {"cfg4": 16, "cfg5": 20, "cfg4s8": 8, "cfg4s10": 10, "cfg4s12": 12, "cfg4h": 32}[name]
        U = _poly_modes([1.0, 0.5, 0.25], g4=[0.03, 0.03, 0.03])
        for a in range(3):
            for b in range(3):
                if a != b:
                    e = [0, 0, 0]
                    e[a] += 1
                    e[b] += 2
                    U.append((0.05 / 6.0, tuple(e)))
        c = dict(n_modes=3, U=U, V_LL=[1.0] * 3, V_SL=[0.2] * 3, zeta=[1.0, 0.65, 0.3], gamma=[0.5, 1.0, 2.0],
                 beta=1.0, depth=3, dt=1e-3, steps=10000, **_grid(3, n, 6.0))
        if name == "cfg4h":     # config 4's model in the Hermite representation (row f1): 32^3 q mesh, np = 8 Hermite
            c["np"] = [8, 8, 8]  # functions per mode -> 20 x 512 x 32768 = 3.36e8 values, the value count of config 4
    else:
        raise KeyError(name)
    c["name"] = name
    c.setdefault("scheme", "central4")
    c.setdefault("gauge", "sqrt_eq")
    c.setdefault("mass", [1.0] * c["n_modes"])
    c.update(over)
    return c


def observable(kind, M):
    """Plain coefficient dicts: mu = sum q_s ; alpha = sum q_s^2 (quad_ss = 2) ; cfg2's mu = q + 0.1 q^2."""
    if kind == "mu":
        return dict(c0=0.0, lin_q=[1.0] * M, quad=[[0.0] * M for _ in range(M)], lin_p=[0.0] * M)
    if kind == "alpha":
        return dict(c0=0.0, lin_q=[0.0] * M, quad=[[2.0 if a == b else 0.0 for b in range(M)] for a in range(M)],
                    lin_p=[0.0] * M)
    if kind == "mu_nl":
        return dict(c0=0.0, lin_q=[1.0] * M, quad=[[0.2 if a == b else 0.0 for b in range(M)] for a in range(M)],
                    lin_p=[0.0] * M)
    if kind == "one":
        return dict(c0=1.0, lin_q=[0.0] * M, quad=[[0.0] * M for _ in range(M)], lin_p=[0.0] * M)
    raise KeyError(kind)


def grid_shape(cfg):
    return tuple(x for s in range(cfg["n_modes"]) for x in (cfg["nq"][s], cfg["np"][s]))


def seeded_state(cfg, levels, seed):
    """Random smooth state exercising every element: X_k = E * 2^-level_k * (1 + 0.5 u), u ~ U(-1,1).

    E is a plain Gaussian envelope exp(-x.x/4) in the grid coordinates (an input distribution, not the
    method's equilibrium).  ``levels`` = |n(k)| per element, as reported by whichever library is fed.
    Canonical layout (K, nq1, np1, ..., nqM, npM), float64.
    """
    rng = np.random.default_rng(seed)
    shape = grid_shape(cfg)
    M = cfg["n_modes"]
    env = np.ones(shape)
    for s in range(M):
        for ax, (lo, hi, n) in ((2 * s, (cfg["qmin"][s], cfg["qmax"][s], cfg["nq"][s])),
                                (2 * s + 1, (cfg["pmin"][s], cfg["pmax"][s], cfg["np"][s]))):
            x = np.linspace(lo, hi, n)
            sh = [1] * len(shape)
            sh[ax] = n
            env = env * np.exp(-0.25 * x * x).reshape(sh)
    X = np.empty((len(levels),) + shape)
    for k, lev in enumerate(levels):
        u = rng.uniform(-1.0, 1.0, size=shape)
        X[k] = env * (0.5 ** lev) * (1.0 + 0.5 * u)
    return X


def seeded_hermite_state(cfg, levels, seed):
    """Random state for the Hermite representation, shape (K, kp_1..kp_M, nq_1..nq_M) with cfg["np"] = Hermite
    functions per mode: c = E(q) * 2^-level * prod_s 0.8^k_s * (1 + 0.5 u), u ~ U(-1,1), E the Gaussian envelope
    exp(-q.q/4).  Exercises every element, every Hermite index and every coupling."""
    rng = np.random.default_rng(seed)
    M = cfg["n_modes"]
    kp, nq = list(cfg["np"][:M]), list(cfg["nq"][:M])
    shape = tuple(kp) + tuple(nq)
    env = np.ones(shape)
    for s in range(M):
        sh = [1] * (2 * M)
        sh[s] = kp[s]
        env = env * (0.8 ** np.arange(kp[s])).reshape(sh)
        x = np.linspace(cfg["qmin"][s], cfg["qmax"][s], nq[s])
        sh = [1] * (2 * M)
        sh[M + s] = nq[s]
        env = env * np.exp(-0.25 * x * x).reshape(sh)
    X = np.empty((len(levels),) + shape)
    for k, lev in enumerate(levels):
        X[k] = env * (0.5 ** lev) * (1.0 + 0.5 * rng.uniform(-1.0, 1.0, size=shape))
    return X

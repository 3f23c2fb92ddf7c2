"""CPU oracle of the Hermite-in-momentum representation (row f1 of DESIGN.md) -- TEST INFRASTRUCTURE, like the rest of
oracle/: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import it.  Plain numpy, fp64; shares
no code with the CUDA path (nor with oracle/chfpe_ref.c).

Eq. (22)-(23) PAPER.md:156-164:  W^(n)(p, q) = prod_s psi_0(p_s) e^{-beta U(q)/2} sum_k c^(n)_k(q) prod_s psi_{k_s}(p_s),
psi_j the orthonormal Hermite functions of width a_s = sqrt(2 m_s / beta).  Since prod psi_0 e^{-beta U/2} is
sqrt(W_eq) up to a constant, sum_k c_k psi_k is the sqrt(W_eq)-gauge variable f of the grid path, and projecting its
equation of motion (reading R1 for the n_s factor) on psi_k with
    p psi_k = a [ sqrt((k+1)/2) psi_{k+1} + sqrt(k/2) psi_{k-1} ],   d/dp psi_k = (1/a) [ sqrt(k/2) psi_{k-1} - sqrt((k+1)/2) psi_{k+1} ]
gives the de-garbled Eq. (A1)-(A4) PAPER.md:343-355 (reading R19; the printed first term and the signs / gamma
factors of Theta, Phi are not consistent with Eq. 8-12):

    d/dt c^(n)_k = sum_s [ sqrt(k_s+1) D+_s c^(n)_{k+e_s} - sqrt(k_s) D-_s c^(n)_{k-e_s} ] - Gamma_n c^(n)_k
                 + sum_s [ n_s gamma_s zeta_s sqrt(m_s/beta) sqrt(k_s+1) V'_s c^(n-e_s)_{k+e_s}
                           - sqrt(k_s beta/m_s) V'_s c^(n+e_s)_{k-e_s} ]
    D+-_s g = (dU/dq_s) / (2 sqrt(m_s/beta)) g  -+  (1/sqrt(m_s beta)) dg/dq_s                      (A2)

with c_k = 0 outside 0 <= k_s < K_p,s and outside the hierarchy simplex (R5), q-derivatives by the CENTRAL4 /
CENTRAL2 stencil with zero ghosts (R9) or by the paper's sixth-order compact scheme (scheme "compact6", Eq. 25-31:
one tridiagonal solve per q-line, here scipy.linalg.solve_banded).  Kick (Eq. 18): c_k <- sum_s (dX/dq_s) (-sqrt(k_s beta/m_s)) c_{k-e_s}.
Expectations: int int O W^(0) dp dq = int O(q) e^{-beta U/2} c^(0)_0(q) dq;  <p_s> uses c^(0)_{e_s} sqrt(m_s/beta).
Equilibrium: c^(0)_0 = e^{-beta U/2} / Z_q, everything else zero.  Time stepping: textbook RK4.
State layout: c[element][k_1]..[k_M][i_q1]..[i_qM].
"""
import itertools

import numpy as np
import scipy.linalg


def enumerate_elements(M, depth):
    """All n in N^M with sum(n) <= depth; ascending |n|, ties by descending lexicographic order (R5, R6)."""
    els = [n for n in itertools.product(range(depth + 1), repeat=M) if sum(n) <= depth]
    els.sort(key=lambda n: (sum(n), tuple(-x for x in n)))
    return els


class RefHermite:
    def __init__(self, cfg):
        self.M = M = cfg["n_modes"]
        self.nq = list(cfg["nq"][:M])
        self.kp = list(cfg["np"][:M])                 # Hermite functions per mode
        self.mass = list(cfg.get("mass", [1.0] * M))[:M]
        self.beta = cfg["beta"]
        self.zeta, self.gamma = list(cfg["zeta"][:M]), list(cfg["gamma"][:M])
        self.VLL, self.VSL = list(cfg["V_LL"][:M]), list(cfg["V_SL"][:M])
        self.scheme = cfg.get("scheme", "central4")
        self.h = [(cfg["qmax"][s] - cfg["qmin"][s]) / (self.nq[s] - 1) for s in range(M)]
        self.q = [cfg["qmin"][s] + self.h[s] * np.arange(self.nq[s]) for s in range(M)]
        self.elems = enumerate_elements(M, cfg["depth"])
        self.K = len(self.elems)
        self.index = {n: k for k, n in enumerate(self.elems)}
        Q = np.meshgrid(*self.q, indexing="ij")
        self.U = np.zeros(self.nq)
        self.dU = [np.zeros(self.nq) for _ in range(M)]
        for coef, expo in cfg["U"]:
            expo = list(expo[:M])
            self.U += coef * np.prod([Q[s] ** expo[s] for s in range(M)], axis=0)
            for s in range(M):
                if expo[s] > 0:
                    e2 = list(expo); e2[s] -= 1
                    self.dU[s] += coef * expo[s] * np.prod([Q[r] ** e2[r] for r in range(M)], axis=0)
        self.Vp = [self.VLL[s] + self.VSL[s] * Q[s] for s in range(M)]
        self.Q = Q
        self.dV = float(np.prod(self.h))
        self.shape = (self.K,) + tuple(self.kp) + tuple(self.nq)
        self.c = np.zeros(self.shape)

    # ---- pieces of the right-hand side -------------------------------------------------------------------------
    def dq(self, g, s):
        """CENTRAL4 / CENTRAL2 derivative along q_s (array axes: k_1..k_M, q_1..q_M), zero ghosts."""
        ax = self.M + s
        n, h = self.nq[s], self.h[s]
        pad = [(0, 0)] * g.ndim
        pad[ax] = (2, 2)
        gp = np.pad(g, pad)
        sl = lambda o: tuple(slice(2 + o, 2 + o + n) if a == ax else slice(None) for a in range(g.ndim))
        if self.scheme == "central2":
            return (gp[sl(1)] - gp[sl(-1)]) / (2 * h)
        if self.scheme == "compact6":
            # Pade scheme of Eq. (25)-(31) PAPER.md:177-201, the paper's q-derivative in this representation:
            # (1/3) d_{i-1} + d_i + (1/3) d_{i+1} = [a (g_{i+1} - g_{i-1}) + b (g_{i+2} - g_{i-2})] / h, a = 7/9 (reading R4:
            # the printed 7/18 is not consistent), b = 1/36, both matrices truncated as printed in Eq. (28)-(29) (R9).
            r = ((7.0 / 9.0) * (gp[sl(1)] - gp[sl(-1)]) + (1.0 / 36.0) * (gp[sl(2)] - gp[sl(-2)])) / h
            ab = np.ones((3, n))
            ab[0, :], ab[2, :] = 1.0 / 3.0, 1.0 / 3.0
            r = np.moveaxis(r, ax, 0)
            d = scipy.linalg.solve_banded((1, 1), ab, r.reshape(n, -1)).reshape(r.shape)
            return np.moveaxis(d, 0, ax)
        return (8.0 * (gp[sl(1)] - gp[sl(-1)]) - (gp[sl(2)] - gp[sl(-2)])) / (12 * h)

    def shift_k(self, g, s, d):
        """Array whose entry k holds g at k + d e_s (zero outside 0 <= k_s < K_p)."""
        out = np.zeros_like(g)
        n = self.kp[s]
        src = [slice(None)] * g.ndim
        dst = [slice(None)] * g.ndim
        if d == 1:
            src[s], dst[s] = slice(1, n), slice(0, n - 1)
        else:
            src[s], dst[s] = slice(0, n - 1), slice(1, n)
        out[tuple(dst)] = g[tuple(src)]
        return out

    def ksqrt(self, s, plus):
        """sqrt(k_s + 1) or sqrt(k_s) broadcast over the element's array."""
        k = np.arange(self.kp[s], dtype=np.float64)
        v = np.sqrt(k + 1.0) if plus else np.sqrt(k)
        shp = [1] * (2 * self.M)
        shp[s] = self.kp[s]
        return v.reshape(shp)

    def rhs(self, c):
        F = np.zeros_like(c)
        M, beta = self.M, self.beta
        for e, n in enumerate(self.elems):
            acc = -sum(n[s] * self.gamma[s] for s in range(M)) * c[e]
            for s in range(M):
                m = self.mass[s]
                up, dn = self.shift_k(c[e], s, +1), self.shift_k(c[e], s, -1)
                a1, a2 = self.dU[s] / (2.0 * np.sqrt(m / beta)), 1.0 / np.sqrt(m * beta)
                acc = acc + self.ksqrt(s, True) * (a1 * up - a2 * self.dq(up, s))        # sqrt(k+1) D+ c_{k+1}
                acc = acc - self.ksqrt(s, False) * (a1 * dn + a2 * self.dq(dn, s))       # sqrt(k)   D- c_{k-1}
                if n[s] > 0:
                    nd = list(n); nd[s] -= 1
                    cd = self.shift_k(c[self.index[tuple(nd)]], s, +1)
                    acc = acc + n[s] * self.gamma[s] * self.zeta[s] * np.sqrt(m / beta) * self.ksqrt(s, True) * self.Vp[s] * cd
                nu = list(n); nu[s] += 1
                if tuple(nu) in self.index:
                    cu = self.shift_k(c[self.index[tuple(nu)]], s, -1)
                    acc = acc - np.sqrt(beta / m) * self.ksqrt(s, False) * self.Vp[s] * cu
            F[e] = acc
        return F

    # ---- protocol --------------------------------------------------------------------------------------------
    def equilibrate(self):
        w = np.exp(-self.beta * self.U)
        self.c[:] = 0.0
        self.c[(0,) + (0,) * self.M] = np.exp(-0.5 * self.beta * self.U) / (np.sum(w) * self.dV)
        F = self.rhs(self.c)
        return float(np.linalg.norm(F) / np.linalg.norm(self.c))

    def step(self, n_steps, dt):
        for _ in range(int(n_steps)):
            y = self.c
            k1 = self.rhs(y)
            k2 = self.rhs(y + 0.5 * dt * k1)
            k3 = self.rhs(y + 0.5 * dt * k2)
            k4 = self.rhs(y + dt * k3)
            self.c = y + (dt / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)

    def _grad(self, obs, s):
        g = obs["lin_q"][s] * np.ones(self.nq)
        for r in range(self.M):
            g = g + 0.5 * (obs["quad"][s][r] + obs["quad"][r][s]) * self.Q[r]
        return g

    def kick(self, obs):
        out = np.zeros_like(self.c)
        for s in range(self.M):
            f = -np.sqrt(self.beta / self.mass[s]) * self._grad(obs, s)
            for e in range(self.K):
                out[e] += f * self.ksqrt(s, False) * self.shift_k(self.c[e], s, -1)
        self.c = out

    def expect(self, obs, element=0):
        w = np.exp(-0.5 * self.beta * self.U)
        O = obs["c0"] * np.ones(self.nq)
        for s in range(self.M):
            O = O + obs["lin_q"][s] * self.Q[s]
            for r in range(self.M):
                O = O + 0.5 * obs["quad"][s][r] * self.Q[s] * self.Q[r]
        val = np.sum(O * w * self.c[(element,) + (0,) * self.M])
        for s in range(self.M):
            if obs["lin_p"][s] != 0.0 and self.kp[s] > 1:
                k1 = [0] * self.M; k1[s] = 1
                val += obs["lin_p"][s] * np.sqrt(self.mass[s] / self.beta) * np.sum(w * self.c[(element,) + tuple(k1)])
        return float(val * self.dV)

    def response_1d(self, A, Cobs, n_samples, stride, dt):
        """Literal Eq. (15): kick A, then <C> every `stride` steps."""
        self.kick(A)
        R = np.empty(n_samples)
        for i in range(n_samples):
            R[i] = self.expect(Cobs)
            if i + 1 < n_samples:
                self.step(stride, dt)
        return R

    def response_2d(self, A, B, Cobs, t1_steps, t2_steps, dt):
        """Literal Eq. (16), the double loop of section IV.C.2 :235-237: the A-kicked state is
        advanced along t1; at every t1 sample a copy gets the B kick and is advanced along t2, <C> recorded."""
        self.kick(A)
        R = np.empty((len(t1_steps), len(t2_steps)))
        now1 = 0
        for i, s1 in enumerate(t1_steps):
            self.step(s1 - now1, dt)
            now1 = s1
            saved = self.c.copy()
            self.kick(B)
            now2 = 0
            for j, s2 in enumerate(t2_steps):
                self.step(s2 - now2, dt)
                now2 = s2
                R[i, j] = self.expect(Cobs)
            self.c = saved
        return R

    def response_3d(self, A, B, Cobs, D, t1_steps, t2_steps, t3_steps, dt):
        """Literal Eq. (17) PAPER.md:126-127 (section IV.C.3 :239-241): R[k][j][l] = <D> after kick A, t1_k, kick B, t2_j,
        kick C, t3_l; plain triple loop with the two trajectories saved and restored."""
        self.kick(A)
        R = np.empty((len(t1_steps), len(t2_steps), len(t3_steps)))
        now1 = 0
        for k, s1 in enumerate(t1_steps):
            self.step(s1 - now1, dt)
            now1 = s1
            T1 = self.c.copy()
            self.kick(B)
            now2 = 0
            for j, s2 in enumerate(t2_steps):
                self.step(s2 - now2, dt)
                now2 = s2
                T2 = self.c.copy()
                self.kick(Cobs)
                now3 = 0
                for l, s3 in enumerate(t3_steps):
                    self.step(s3 - now3, dt)
                    now3 = s3
                    R[k, j, l] = self.expect(D)
                self.c = T2
            self.c = T1
        return R

    def export_state(self):
        return self.c.copy()

    def import_state(self, c):
        self.c = np.array(c, dtype=np.float64).reshape(self.shape)

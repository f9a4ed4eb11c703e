"""Third, even more literal evaluator of the TSLB step for tiny periodic grids (pin P10).

Independent of oracle/ and of the CUDA path: numpy only, full (non-deviation) populations, the
non-equilibrium Hermite coefficient obtained by PROJECTION (eq. 14) of f - f^eq rather
than from the stored moments, every tensor contraction written as an explicit einsum over all 27
velocities and all alpha,beta,gamma (eq. 16, 183 eq. 19), g populations of the D3Q7
phase-field LB formed explicitly (eqs. 23-24).
"""
import itertools

import numpy as np

CS2 = 1.0 / 3.0


def d3q27():
    c = np.array(list(itertools.product((-1, 0, 1), repeat=3)), dtype=np.int64)  # any order
    w1 = {0: 2.0 / 3.0, 1: 1.0 / 6.0, -1: 1.0 / 6.0}
    w = np.array([w1[a] * w1[b] * w1[g] for a, b, g in c])
    return c, w


def hermite(c):
    cf = c.astype(np.float64)
    d = np.eye(3)
    H2 = np.einsum("ia,ib->iab", cf, cf) - CS2 * d[None]
    H3 = (np.einsum("ia,ib,ig->iabg", cf, cf, cf)
          - CS2 * (np.einsum("ig,ab->iabg", cf, d) + np.einsum("ia,bg->iabg", cf, d)
                   + np.einsum("ib,ag->iabg", cf, d)))
    return H2, H3


def shift(a, cvec):
    """value at x - c  ->  roll by +c along (z,y,x) axes of an array (..., nz, ny, nx)."""
    return np.roll(a, shift=(int(cvec[2]), int(cvec[1]), int(cvec[0])), axis=(-3, -2, -1))


class BruteForce:
    def __init__(self, omega, sigma=0.0, W=4.0, two=True, order=3, guo=False):
        self.guo = guo
        self.c, self.w = d3q27()
        self.H2, self.H3 = hermite(self.c)
        self.omega, self.sigma, self.gamma, self.two, self.order = omega, sigma, 2.0 / W, two, order
        self.c7 = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1],
                            [0, 0, -1]])
        self.w7 = np.array([0.25] + [0.125] * 6)

    def feq(self, rho, u):
        """eq. 16; rho (...), u (3, ...) -> (27, ...)"""
        cf = self.c.astype(np.float64)
        t1 = np.einsum("ia,a...->i...", cf, u) / CS2
        t2 = np.einsum("iab,a...,b...->i...", self.H2, u, u) / (2 * CS2 ** 2)
        t3 = np.einsum("iabg,a...,b...,g...->i...", self.H3, u, u, u) / (6 * CS2 ** 3)
        if self.order < 3:
            t3 = 0.0
        return self.w.reshape((27,) + (1,) * rho.ndim) * rho[None] * (1.0 + t1 + t2 + t3)

    def fneq_reg(self, a2, u):
        """eq. 19 (Hermite form: w_i prefactor, H2 = cc - cs2 delta); a2 (3,3,...), u (3,...)"""
        a3 = (np.einsum("ab...,g...->abg...", a2, u) + np.einsum("a...,bg...->abg...", u, a2)
              + np.einsum("b...,ag...->abg...", u, a2))
        t2 = np.einsum("iab,ab...->i...", self.H2, a2) / (2 * CS2 ** 2)
        t3 = np.einsum("iabg,abg...->i...", self.H3, a3) / (6 * CS2 ** 3)
        if self.order < 3:
            t3 = 0.0
        return self.w.reshape((27,) + (1,) * (u.ndim - 1)) * (t2 + t3)

    def init(self, rho, u, phi, pineq6):
        a2 = self._sym(pineq6)
        self.u = u.copy()
        self.phi = None if phi is None else phi.copy()
        if self.guo:
            # full second moment of the given state, then the Guo collision with F(phi(0))
            Pfull = a2 + rho[None, None] * (CS2 * np.eye(3)[:, :, None, None, None]
                                             + np.einsum("a...,b...->ab...", u, u))
            self.rho = rho.copy()
            F = self._force(self.phi)[0]
            m = rho[None] * u
            uc = (m + 0.5 * F) / rho[None]                               # Guo: rho u = m + F/2
            a2c = Pfull - rho[None, None] * (CS2 * np.eye(3)[:, :, None, None, None]
                                             + np.einsum("a...,b...->ab...", uc, uc))
            self.f = self._collide_guo(rho, uc, m - rho[None] * uc, a2c, F)
            return
        self.f = self.feq(rho, u) + (1 - self.omega) * self.fneq_reg(a2, u)

    # ---- reading A18: forcing of Guo, Zheng & Shi (2002), written from the published scheme with
    # the pre-collision populations regularised by projection (eq. 14) up to third order
    def _force(self, phi):
        c, w = self.c, self.w
        cf = c.astype(np.float64)
        G = np.zeros((3,) + phi.shape)
        for i in range(27):
            G += w[i] * cf[i][:, None, None, None] * shift(phi, -c[i])[None]
        G /= CS2
        n = G / (np.sqrt((G * G).sum(0)) + 1e-12)
        div = np.zeros_like(phi)
        for i in range(27):
            div += w[i] * np.einsum("a,a...->...", cf[i], shift(n, -c[i]))
        return self.sigma * (-div / CS2)[None] * G, n

    def _collide_guo(self, rho, u, a1, a2, F):
        """rho, collision velocity u, first and second Hermite moments a1, a2 of f - f^eq(rho,u),
        force F -> f^post = f^eq + (1-omega)(f^pre - f^eq) + (1-omega/2) S."""
        cf = self.c.astype(np.float64)
        feq = self.feq(rho, u)
        wsh = self.w.reshape((27, 1, 1, 1))
        fpre = feq + self.fneq_reg(a2, u) + wsh * np.einsum("ia,a...->i...", cf, a1) / CS2
        cF = np.einsum("ia,a...->i...", cf, F)
        cu = np.einsum("ia,a...->i...", cf, u)
        uF = (u * F).sum(0)[None]
        S = wsh * ((cF - uF) / CS2 + cu * cF / CS2 ** 2)
        return feq + (1 - self.omega) * (fpre - feq) + (1 - 0.5 * self.omega) * S

    def step_guo(self):
        c = self.c
        cf = c.astype(np.float64)
        F_old, n_old = self._force(self.phi)
        u_phys = self.u + 0.5 * F_old / self.rho[None]
        f = np.stack([shift(self.f[i], c[i]) for i in range(27)])
        rho = f.sum(0)
        m = np.einsum("ia,i...->a...", cf, f)
        Pfull = np.einsum("ia,ib,i...->ab...", cf, cf, f)
        f_streamed = f
        phi = self.phi
        gpost = []
        for q in range(7):
            cq = self.c7[q].astype(np.float64)
            cu = np.einsum("a,a...->...", cq, u_phys)
            cn = np.einsum("a,a...->...", cq, n_old)
            gpost.append(self.w7[q] * phi * (1 + cu / 0.25) + self.w7[q] * self.gamma * phi * (1 - phi) * cn)
        self.phi = sum(shift(gpost[q], self.c7[q]) for q in range(7))
        F = self._force(self.phi)[0]
        uc = (m + 0.5 * F) / rho[None]                                   # Guo: rho u = m + F/2
        fneq_pre = f_streamed - self.feq(rho, uc)                        # eq. 14, projection
        self.f = self._collide_guo(rho, uc, np.einsum("ia,i...->a...", cf, fneq_pre),
                                   np.einsum("iab,i...->ab...", self.H2, fneq_pre), F)
        ub = m / rho[None]
        a2b = Pfull - rho[None, None] * (CS2 * np.eye(3)[:, :, None, None, None] + np.einsum("a...,b...->ab...", ub, ub))
        self.u, self.rho = ub, rho
        self.pineq6 = np.stack([a2b[0, 0], a2b[1, 1], a2b[2, 2], a2b[0, 1], a2b[0, 2], a2b[1, 2]])

    @staticmethod
    def _sym(p6):
        a = np.empty((3, 3) + p6.shape[1:])
        a[0, 0], a[1, 1], a[2, 2] = p6[0], p6[1], p6[2]
        a[0, 1] = a[1, 0] = p6[3]
        a[0, 2] = a[2, 0] = p6[4]
        a[1, 2] = a[2, 1] = p6[5]
        return a

    def step(self):
        if self.guo:
            return self.step_guo()
        c, w = self.c, self.w
        cf = c.astype(np.float64)
        f = np.stack([shift(self.f[i], c[i]) for i in range(27)])          # eq. 1 / eq. 6
        rho = f.sum(0)
        ub = np.einsum("ia,i...->a...", cf, f) / rho
        unew = ub.copy()
        if self.two:
            phi = self.phi
            G = np.zeros_like(ub)
            for i in range(27):
                G += w[i] * cf[i][:, None, None, None] * shift(phi, -c[i])[None]   # phi(x + c_i)
            G /= CS2
            n = G / (np.sqrt((G * G).sum(0)) + 1e-12)
            div = np.zeros_like(phi)
            for i in range(27):
                div += w[i] * np.einsum("a,a...->...", cf[i], shift(n, -c[i]))
            kappa = -div / CS2
            unew = ub + self.sigma * kappa[None] * G / rho[None]
            # D3Q7 populations after "collision" (unit relaxation time): g^eq + Lambda
            gpost = []
            for q in range(7):
                cq = self.c7[q].astype(np.float64)
                cu = np.einsum("a,a...->...", cq, self.u)
                cn = np.einsum("a,a...->...", cq, n)
                gpost.append(self.w7[q] * phi * (1 + cu / 0.25) + self.w7[q] * self.gamma * phi * (1 - phi) * cn)
            self.phi = sum(shift(gpost[q], self.c7[q]) for q in range(7))
        fneq_pre = f - self.feq(rho, ub)
        a2 = np.einsum("iab,i...->ab...", self.H2, fneq_pre)              # eq. 14, projection
        self.f = self.feq(rho, unew) + (1 - self.omega) * self.fneq_reg(a2, unew)
        self.u = unew
        self.rho = rho
        self.pineq6 = np.stack([a2[0, 0], a2[1, 1], a2[2, 2], a2[0, 1], a2[0, 2], a2[1, 2]])

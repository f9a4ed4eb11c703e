"""Pins P1-P3 (+ the A3/A4/A17 readings): the oracle's lattice, equilibrium and regularized
non-equilibrium against what the paper and the mathematics fix.  CPU only."""
import itertools

import numpy as np
import pytest

from oracle import ref

CS2 = 1.0 / 3.0
rng = np.random.default_rng(20240315)


def test_p1_lattice_identities():
    """PAPER.md:79 ("normalized set of weights", c_s^2 = 1/3), 116 Fig. 2 (three speed groups)."""
    c, w = ref.lattice()
    assert sorted(map(tuple, c.tolist())) == sorted(itertools.product((-1, 0, 1), repeat=3))
    speed2 = (c * c).sum(1)
    for s2, wv, cnt in ((0, 8 / 27, 1), (1, 2 / 27, 6), (2, 1 / 54, 12), (3, 1 / 216, 8)):
        assert (speed2 == s2).sum() == cnt
        np.testing.assert_allclose(w[speed2 == s2], wv, rtol=1e-15)
    cf = c.astype(float)
    d = np.eye(3)
    assert abs(w.sum() - 1) < 1e-15
    np.testing.assert_allclose(np.einsum("i,ia->a", w, cf), 0, atol=1e-16)
    np.testing.assert_allclose(np.einsum("i,ia,ib->ab", w, cf, cf), CS2 * d, atol=1e-16)
    np.testing.assert_allclose(np.einsum("i,ia,ib,ig->abg", w, cf, cf, cf), 0, atol=1e-16)
    iso4 = CS2 ** 2 * (np.einsum("ab,gd->abgd", d, d) + np.einsum("ag,bd->abgd", d, d)
                       + np.einsum("ad,bg->abgd", d, d))
    np.testing.assert_allclose(np.einsum("i,ia,ib,ig,id->abgd", w, cf, cf, cf, cf), iso4, atol=1e-16)
    # 1-D tensor-product basis {1, c, c^2 - 1/3}: orthogonal with norms 1, 1/3, 2/9
    w1 = np.array([1 / 6, 2 / 3, 1 / 6]); s = np.array([-1.0, 0.0, 1.0])
    h = np.stack([np.ones(3), s, s * s - CS2])
    np.testing.assert_allclose(np.einsum("s,as,bs->ab", w1, h, h), np.diag([1, 1 / 3, 2 / 9]), atol=1e-16)


def _rand_state():
    rho = 1 + 0.05 * rng.uniform(-1, 1)
    u = 0.1 * rng.uniform(-1, 1, 3)
    p6 = 5e-3 * rng.uniform(-1, 1, 6)
    return rho, u, p6


def _sym(p6):
    return np.array([[p6[0], p6[3], p6[4]], [p6[3], p6[1], p6[5]], [p6[4], p6[5], p6[2]]])


@pytest.mark.parametrize("order", [2, 3])
def test_p2_rebuilt_populations_carry_the_stored_moments(order):
    """f rebuilt from (rho, u, Pi^neq) has moments rho, rho u,
    rho u u + rho c_s^2 delta + (1-omega) Pi^neq.  Fails for the literal (garbled) eq. 19 (A3)."""
    c, w = ref.lattice()
    cf = c.astype(float)
    for _ in range(20):
        rho, u, p6 = _rand_state()
        omega = rng.uniform(0.3, 1.99)
        fe, fn = ref.feq(rho, u, order), ref.fneq(p6, u, order)
        f = fe + (1 - omega) * fn
        assert abs(f.sum() - rho) < 2e-16 * 10
        np.testing.assert_allclose(cf.T @ f, rho * u, atol=1e-16)
        P = np.einsum("i,ia,ib->ab", f, cf, cf)
        np.testing.assert_allclose(P, rho * np.outer(u, u) + rho * CS2 * np.eye(3) + (1 - omega) * _sym(p6),
                                   atol=3e-16)
        # the collision conserves mass and momentum: sum f^neq = 0, sum c f^neq = 0
        assert abs(fn.sum()) < 1e-17
        np.testing.assert_allclose(cf.T @ fn, 0, atol=1e-17)


def test_p3_third_moment_of_equilibrium():
    """PAPER.md:172 eq. 17: eq. 16 recovers Q_abg = rho u_a u_b u_g + rho c_s^2 (u_a d_bg + ...)
    for every non-(aaa) component (aaa is aliased on {-1,0,1}: c^3 = c)."""
    c, w = ref.lattice()
    cf = c.astype(float)
    d = np.eye(3)
    for _ in range(10):
        rho, u, _ = _rand_state()
        f = ref.feq(rho, u, 3)
        Q = np.einsum("i,ia,ib,ig->abg", f, cf, cf, cf)
        Qx = rho * np.einsum("a,b,g->abg", u, u, u) + rho * CS2 * (
            np.einsum("a,bg->abg", u, d) + np.einsum("b,ag->abg", u, d) + np.einsum("g,ab->abg", u, d))
        for a, b, g in itertools.product(range(3), repeat=3):
            if a == b == g:
                continue
            assert abs(Q[a, b, g] - Qx[a, b, g]) < 1e-16
        # order 2 does NOT recover it (so the pin does discriminate)
        Q2 = np.einsum("i,ia,ib,ig->abg", ref.feq(rho, u, 2), cf, cf, cf)
        assert abs(Q2[0, 0, 1] - Qx[0, 0, 1]) > 1e-6


def test_third_order_hermite_coefficients_of_fneq():
    """PAPER.md:156 eq. 14 applied to eq. 19: projecting f^neq on H^3 must give back
    a^3_abg = Pi_ab u_g + u_a Pi_bg + u_b Pi_ag (pins the 1/(6 c_s^6) factor and the three-term
    recursion, A4) for the non-aliased components; and on H^2 gives Pi^neq (A17)."""
    c, w = ref.lattice()
    cf = c.astype(float)
    d = np.eye(3)
    for _ in range(10):
        _, u, p6 = _rand_state()
        a2 = _sym(p6)
        fn = ref.fneq(p6, u, 3)
        H2 = np.einsum("ia,ib->iab", cf, cf) - CS2 * d[None]
        np.testing.assert_allclose(np.einsum("i,iab->ab", fn, H2), a2, atol=1e-17)
        H3 = (np.einsum("ia,ib,ig->iabg", cf, cf, cf) - CS2 * (
            np.einsum("ig,ab->iabg", cf, d) + np.einsum("ia,bg->iabg", cf, d) + np.einsum("ib,ag->iabg", cf, d)))
        a3 = np.einsum("i,iabg->abg", fn, H3)
        a3x = (np.einsum("ab,g->abg", a2, u) + np.einsum("a,bg->abg", u, a2) + np.einsum("b,ag->abg", u, a2))
        for a, b, g in itertools.product(range(3), repeat=3):
            if a == b == g:
                assert abs(a3[a, b, g]) < 1e-17       # H3_aaa == 0 on this lattice
            else:
                assert abs(a3[a, b, g] - a3x[a, b, g]) < 1e-17


def test_order2_is_eq8():
    """hermite_order = 2 must be PAPER.md:120 eq. 8 term by term (eq. 2 + eq. 7)."""
    c, w = ref.lattice()
    cf = c.astype(float)
    for _ in range(10):
        rho, u, p6 = _rand_state()
        cu = cf @ u
        eq2 = w * rho * (1 + cu / CS2 + (cu * cu - CS2 * (u @ u)) / (2 * CS2 ** 2))
        ccP = np.einsum("ia,ab,ib->i", cf, _sym(p6), cf)
        eq7 = w / (2 * CS2 ** 2) * (ccP - CS2 * np.trace(_sym(p6)))
        np.testing.assert_allclose(ref.feq(rho, u, 2), eq2, atol=1e-16)
        np.testing.assert_allclose(ref.fneq(p6, u, 2), eq7, atol=1e-17)


def test_order3_closed_forms():
    """Scalar closed forms of eqs. 16 and 19 (contracting the Hermite tensors by hand):
    f^eq_3 = w rho (c.u)((c.u)^2 - 3 c_s^2 u.u)/(6 c_s^6),
    f^neq_3 = w [(c.Pi.c)(c.u) - c_s^2 (tr Pi (c.u) + 2 c.Pi.u)]/(2 c_s^6)."""
    c, w = ref.lattice()
    cf = c.astype(float)
    for _ in range(10):
        rho, u, p6 = _rand_state()
        P = _sym(p6)
        cu = cf @ u
        t3 = w * rho * cu * (cu * cu - 3 * CS2 * (u @ u)) / (6 * CS2 ** 3)
        np.testing.assert_allclose(ref.feq(rho, u, 3) - ref.feq(rho, u, 2), t3, atol=1e-16)
        cPc = np.einsum("ia,ab,ib->i", cf, P, cf)
        n3 = w * (cPc * cu - CS2 * (np.trace(P) * cu + 2 * cf @ (P @ u))) / (2 * CS2 ** 3)
        np.testing.assert_allclose(ref.fneq(p6, u, 3) - ref.fneq(p6, u, 2), n3, atol=1e-17)


def test_p13_inflow_hash_restated():
    """A12: xi = (2k+1-2^24)/2^24 with k the top 24 bits of the splitmix64 finaliser of
    seed + (counter+1)*golden, counter = step*nx*ny + x + nx*y.  Restated with Python ints."""
    M = (1 << 64) - 1

    def xi_py(seed, x, y, nx, ny, step):
        z = (seed + (step * nx * ny + x + nx * y + 1) * 0x9E3779B97F4A7C15) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        z ^= z >> 31
        return (2 * (z >> 40) + 1 - (1 << 24)) / float(1 << 24)

    vals = []
    for step in (0, 1, 2, 1000, 123456):
        for (x, y) in ((0, 0), (5, 3), (63, 63), (17, 42)):
            v = ref.xi(2024, x, y, 64, 64, step)
            assert v == xi_py(2024, x, y, 64, 64, step)
            assert -1 < v < 1
            vals.append(v)
    assert len(set(vals)) == len(vals)
    big = np.array([ref.xi(7, x, y, 64, 64, 3) for x in range(64) for y in range(64)])
    assert abs(big.mean()) < 0.03 and abs(big.std() - 1 / np.sqrt(3)) < 0.02
    # every value is an odd multiple of 2^-24: exactly representable in fp32
    assert np.all(big.astype(np.float32).astype(np.float64) == big)

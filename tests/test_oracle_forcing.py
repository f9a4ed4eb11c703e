"""Pins of the oracle's second forcing reading A18 (time-centred forcing of Guo,
Zheng & Shi, Phys. Rev. E 65 (2002) 046308) and of the physical-velocity accessor of both
readings.  The paper does not say how F = sigma kappa grad(phi) enters the flow solver
(PAPER.md:188-215), so these pins are what the published forcing scheme and the mathematics fix:
the moment conditions of the forced collision, exact momentum balance, uniform acceleration,
the steady Kolmogorov flow, Young-Laplace, and an independent numpy restatement on 8^3.  CPU only."""
import math

import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import inputs
from tests.brute_force import BruteForce

CS2 = 1.0 / 3.0
GUO, KICK = ref.FORCING_GUO, ref.FORCING_KICK


def _state(o):
    m = o.get_moments()
    return m, np.stack([m["ux"], m["uy"], m["uz"]])


def test_f1_sigma_zero_guo_is_kick_bit_for_bit():
    """With F = 0 the forced collision is the unforced one: both readings then give identical bits."""
    d = inputs.droplets_noise(16, seed=3, ndrop=2, rmin=3.0, rmax=4.0, W=3.0, noise=0.01)
    res = []
    for f in (KICK, GUO):
        o = ref.Oracle(16, 16, 16, 1.7, two_component=True, sigma=0.0, interface_width=3.0, forcing=f)
        o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
        o.step(5)
        res.append(o.get_moments())
    for k in ("rho", "ux", "uy", "uz", "pineq", "phi"):
        assert np.array_equal(res[0][k], res[1][k]), k


@pytest.mark.parametrize("order", [3, 2])
def test_f2_moment_conditions_of_the_forced_collision(order):
    """Guo et al. (2002): the post-collision populations carry mass rho, momentum m + F, and the
    second moment rho c_s^2 delta + rho u u + (1-omega) Pi^neq + (1-omega/2)(uF + Fu) with
    rho u = m + F/2 and Pi^neq = Pi - rho c_s^2 delta - rho u u, which in terms of the stored bare
    moments is Pi_b^neq - (u_b F + F u_b)/2 - F F/(4 rho).
    Third order (eq. 19 recursion): rho u u u + (1-omega)(Pi^neq u)_sym on the components the
    lattice represents.  Checked on the oracle's stored populations for a random state + force."""
    n = 6
    d = inputs.smooth_random(n, n, n, seed=5)
    rng = np.random.default_rng(17)
    Fx = 1e-3 * rng.standard_normal((3, n, n, n))
    omega = 1.6
    o = ref.Oracle(n, n, n, omega, hermite_order=order, forcing=GUO)
    o.set_extra_force(Fx)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], None, d["pineq"])
    f = o.get_populations()
    c, w = ref.lattice()
    cf = c.astype(np.float64)
    rho = d["rho"]
    ub = np.stack([d["ux"], d["uy"], d["uz"]])
    u = ub + Fx / (2 * rho)
    P6 = d["pineq"]
    Pb = np.empty((3, 3, n, n, n))
    for (a, b), k in {(0, 0): 0, (1, 1): 1, (2, 2): 2, (0, 1): 3, (0, 2): 4, (1, 2): 5}.items():
        Pb[a, b] = Pb[b, a] = P6[k]
    ubF = np.einsum("a...,b...->ab...", ub, Fx)
    PG = Pb - 0.5 * (ubF + ubF.transpose(1, 0, 2, 3, 4)) - np.einsum("a...,b...->ab...", Fx, Fx) / (4 * rho)
    assert np.abs(f.sum(0) - rho).max() < 1e-14
    mom = np.einsum("ia,i...->a...", cf, f)
    assert np.abs(mom - (rho * ub + Fx)).max() < 1e-15
    sec = np.einsum("ia,ib,i...->ab...", cf, cf, f)
    uF = np.einsum("a...,b...->ab...", u, Fx)
    want = (rho * (CS2 * np.eye(3)[:, :, None, None, None] + np.einsum("a...,b...->ab...", u, u))
            + (1 - omega) * PG + (1 - omega / 2) * (uF + uF.transpose(1, 0, 2, 3, 4)))
    assert np.abs(sec - want).max() < 1e-15
    assert np.abs((1 - omega / 2) * uF).max() > 1e-6          # the source term is not negligible here
    if order == 3:
        third = np.einsum("ia,ib,ig,i...->abg...", cf, cf, cf, f)
        a3 = (rho * np.einsum("a...,b...,g...->abg...", u, u, u)
              + (1 - omega) * (np.einsum("ab...,g...->abg...", PG, u) + np.einsum("a...,bg...->abg...", u, PG)
                               + np.einsum("b...,ag...->abg...", u, PG)))
        m1 = rho * ub + Fx
        for (a, b, g) in [(0, 0, 1), (0, 0, 2), (1, 1, 0), (1, 1, 2), (2, 2, 0), (2, 2, 1), (0, 1, 2)]:
            # sum c_a c_b c_g f = a3_abg + c_s^2 (first moment)_g delta_ab  (+ perms; here a == b != g or all distinct)
            corr = CS2 * m1[g] if a == b else 0.0
            assert np.abs(third[a, b, g] - (a3[a, b, g] + corr)).max() < 1e-15, (a, b, g)


def test_f3_momentum_balance_and_conservation_guo():
    """Every step adds exactly the force of the time level that was collided: sum m(t+1) - sum m(t)
    = sum F(t); mass and phi are conserved."""
    d = inputs.droplets_noise(20, seed=3, ndrop=3, rmin=3.0, rmax=5.0, W=3.0, noise=0.01)
    o = ref.Oracle(20, 20, 20, 1.7, two_component=True, sigma=0.01, interface_width=3.0, forcing=GUO)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    m0 = o.get_moments()
    for _ in range(20):
        mb = o.get_moments()
        _, _, _, F = o.phase_geometry()
        o.step(1)
        ma = o.get_moments()
        for a, k in enumerate(("ux", "uy", "uz")):
            dp = (ma["rho"] * ma[k]).sum() - (mb["rho"] * mb[k]).sum()
            assert abs(dp - F[a].sum()) < 1e-12
        up = o.get_physical_velocity()
        _, _, _, Fn = o.phase_geometry()
        assert np.abs(up[0] - (ma["ux"] + Fn[0] / (2 * ma["rho"]))).max() < 1e-16
    m1 = o.get_moments()
    assert abs(m1["rho"].sum() / m0["rho"].sum() - 1) < 1e-13
    assert abs(m1["phi"].sum() / m0["phi"].sum() - 1) < 1e-13
    assert np.abs(F).max() > 1e-5


@pytest.mark.parametrize("forcing", [KICK, GUO])
def test_f4_uniform_acceleration(forcing):
    """A uniform force density g on a uniform fluid moving with U: the momentum grows by g per step,
    exactly; the time-centred velocity at step n is U + (n +- 1/2) g / rho (stored state at step n
    is the bare momentum for GUO, the kicked one for KICK); the density stays uniform."""
    n, steps = 6, 40
    g = np.array([3e-5, -2e-5, 1e-5])
    U = np.array([0.03, 0.01, -0.02])
    rho = np.full((n, n, n), 1.0)
    o = ref.Oracle(n, n, n, 1.4, forcing=forcing)
    o.set_extra_force(np.broadcast_to(g[:, None, None, None], (3, n, n, n)).copy())
    o.init_fields(rho, *(np.full((n, n, n), U[a]) for a in range(3)))
    o.step(steps)
    m, u = _state(o)
    up = o.get_physical_velocity()
    assert np.abs(m["rho"] - 1).max() < 1e-14
    for a in range(3):
        assert np.abs(u[a] - (U[a] + steps * g[a])).max() < 1e-15
        half = 0.5 if forcing == GUO else -0.5
        assert np.abs(up[a] - (U[a] + (steps + half) * g[a])).max() < 1e-15
    if forcing == GUO:
        # the second-order source (uF + Fu) keeps the stress at its equilibrium value: the stored
        # Pi_b^neq is O(g^2) (steady value -(1/omega + 1/4) F F/rho); without that source, or with a
        # mis-weighted one, it is O(U g) ~ 1e-6
        assert np.abs(m["pineq"]).max() < 20 * (g ** 2).max()


@pytest.mark.parametrize("forcing", [KICK, GUO])
def test_f5_kolmogorov_flow_steady_state(forcing):
    """F_x = A sin(k y) on a fluid at rest.  For this unidirectional flow the steady state of the
    lattice scheme satisfies the discrete momentum balance  nu k~^2 (m_post / rho) = F / rho  EXACTLY,
    m_post = momentum after the forced collision (the one that is streamed), k~^2 = 2 (1 - cos k)
    (second difference of the streaming step), nu = c_s^2 (1/omega - 1/2) -- in both
    readings, because with u_y = 0 the collision velocity only enters moments the balance does not
    see.  KICK (A9) stores m_post / rho; GUO (A18) stores the bare (m_post - F)/rho.  The time-centred
    velocity of either reading is (m_post - F/2)/rho.  Fixes the unit weight of the force in the
    momentum, the (1 - omega/2) weight of the source against the F/2 in the collision velocity, and
    both accessors.  Gate 1e-9; a mis-weighted force changes the amplitude by O(1)."""
    nx, ny, nz, omega, A = 4, 16, 4, 1.0, 1e-6
    nu = CS2 * (1 / omega - 0.5)
    k = 2 * math.pi / ny
    y = np.arange(ny)
    F = np.zeros((3, nz, ny, nx))
    F[0] = A * np.sin(k * y)[None, :, None]
    one = np.ones((nz, ny, nx))
    o = ref.Oracle(nx, ny, nz, omega, forcing=forcing)
    o.set_extra_force(F)
    o.init_fields(one, 0 * one, 0 * one, 0 * one)
    o.step(1200)                                   # e-folding time 1/(nu k^2) = 39 steps
    up = o.get_physical_velocity()
    _, u = _state(o)
    kt2 = 2 * (1 - math.cos(k))
    amp_phys = (up[0] * F[0]).sum() / (F[0] ** 2).sum() * A
    amp_stored = (u[0] * F[0]).sum() / (F[0] ** 2).sum() * A
    want = A / (nu * kt2)
    amp_post = amp_stored + (A if forcing == GUO else 0.0)
    assert abs(amp_post / want - 1) < 1e-9, amp_post / want
    assert abs((amp_post - amp_phys) / (0.5 * A) - 1) < 1e-9
    assert np.abs(up[1]).max() < 1e-18 and np.abs(up[2]).max() < 1e-18


def test_f6_young_laplace_guo():
    """the forced scheme must reproduce dp = 2 sigma / R whichever way the force enters
    (same droplet and gates as P9: R = 8, W = 4 in 32^3, finite-width excess ~ +4 %)."""
    n, R, W, sigma = 32, 8.0, 4.0, 0.01
    d = inputs.static_droplet(n, R, W)
    o = ref.Oracle(n, n, n, 1.0, two_component=True, sigma=sigma, interface_width=W, forcing=GUO)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    zz, yy, xx = np.meshgrid(*(np.arange(n) - (n - 1) / 2.0,) * 3, indexing="ij")
    r = np.sqrt(xx ** 2 + yy ** 2 + zz ** 2)
    inside, outside = r < R / 2, r > R + 2 * W
    o.step(300)
    dps = []
    for _ in range(111):
        o.step(1)
        m = o.get_moments()
        dps.append(CS2 * (m["rho"][inside].mean() - m["rho"][outside].mean()))
    ratio = float(np.mean(dps)) / (2 * sigma / R)
    assert 1.0 < ratio < 1.06, ratio
    assert np.abs(o.get_physical_velocity()).max() < 2e-4      # spurious currents stay small


@pytest.mark.parametrize("order", [3, 2])
def test_f7_brute_force_8cubed_guo(order):
    """Independent numpy restatement (tests/brute_force.py: full populations, projection route,
    Guo's published collision) against the oracle's A18 step."""
    d = inputs.smooth_random(8, 8, 8, seed=11)
    omega, sigma, W = 1.85, 0.02, 3.0
    o = ref.Oracle(8, 8, 8, omega, two_component=True, sigma=sigma, interface_width=W,
                   hermite_order=order, forcing=GUO)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"], d["pineq"])
    b = BruteForce(omega, sigma, W, two=True, order=order, guo=True)
    b.init(d["rho"], np.stack([d["ux"], d["uy"], d["uz"]]), d["phi"], d["pineq"])
    fo = np.sort(o.get_populations().reshape(27, -1), axis=0)
    fb = np.sort(b.f.reshape(27, -1), axis=0)
    assert np.abs(fo - fb).max() < 1e-15
    for step in range(5):
        o.step(1)
        b.step()
        m = o.get_moments()
        assert np.abs(m["rho"] - b.rho).max() < 1e-13
        for a, k in enumerate(("ux", "uy", "uz")):
            assert np.abs(m[k] - b.u[a]).max() / np.abs(b.u).max() < 1e-13
        assert np.abs(m["pineq"] - b.pineq6).max() / np.abs(b.pineq6).max() < 1e-12
        assert np.abs(m["phi"] - b.phi).max() < 1e-13
    _, _, _, F = o.phase_geometry()
    assert np.abs(F).max() > 1e-5 and np.abs(b.u).max() > 1e-3

"""Pins P4-P12 of the CPU oracle: conservation, closed-form decay rates, fixed points, exact
one-step amplification of the D3Q7 phase step, stationary planar interface, Young-Laplace,
8^3 brute force, lattice equivariance, stencil exactness, jet boundary sanity.  CPU only."""
import math

import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import inputs
from tests.brute_force import BruteForce

CS2 = 1.0 / 3.0


def _run(d, omega, steps, **kw):
    nz, ny, nx = d["rho"].shape
    o = ref.Oracle(nx, ny, nz, omega, two_component=d.get("phi") is not None, **kw)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
    o.step(steps)
    return o


# ---------------------------------------------------------------- P4 conservation
def test_p4_mass_phi_conserved_and_momentum_balance():
    """PAPER.md:71 eq. 1 conserves mass and momentum; eqs. 23-24 conserve phi (sum_i Lambda_i = 0);
    the kick (A9) adds exactly F per node per step."""
    d = inputs.droplets_noise(20, seed=3, ndrop=3, rmin=3.0, rmax=5.0, W=3.0, noise=0.01)
    o = ref.Oracle(20, 20, 20, 1.7, two_component=True, sigma=0.01, interface_width=3.0)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    m0 = o.get_moments()
    mass0, phi0 = m0["rho"].sum(), m0["phi"].sum()
    for _ in range(30):
        mb = o.get_moments()
        _, _, _, F = o.phase_geometry()          # force from the time-t phi
        o.step(1)
        ma = o.get_moments()
        for a, k in enumerate(("ux", "uy", "uz")):
            dp = (ma["rho"] * ma[k]).sum() - (mb["rho"] * mb[k]).sum()
            assert abs(dp - F[a].sum()) < 1e-12
    m1 = o.get_moments()
    assert abs(m1["rho"].sum() - mass0) / mass0 < 1e-13
    assert abs(m1["phi"].sum() - phi0) / phi0 < 1e-13
    assert np.abs(F).max() > 1e-5               # the balance was not trivially 0 = 0


# ---------------------------------------------------------------- P5 viscosity
@pytest.mark.parametrize("axis,shape", [("y", (4, 32, 4)), ("z", (4, 4, 32))])
@pytest.mark.parametrize("omega", [0.8, 1.8])
def test_p5_shear_wave_decay(axis, shape, omega):
    """nu = c_s^2 (1/omega - 1/2); u_x = U0 sin(k s) decays as exp(-nu k^2 t)."""
    nx, ny, nz = shape
    d = inputs.shear_wave(nx, ny, nz, 0.01, axis)
    o = ref.Oracle(nx, ny, nz, omega)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"])
    amp = []
    for _ in range(201):
        m = o.get_moments()
        amp.append((m["ux"] * d["ux"]).sum() / (d["ux"] ** 2).sum())
        o.step(1)
    nu = CS2 * (1 / omega - 0.5)
    k = 2 * math.pi / 32
    rate = -np.polyfit(np.arange(40, 201), np.log(np.array(amp[40:201])), 1)[0]
    assert abs(rate / (nu * k * k) - 1) < 5e-3


@pytest.mark.parametrize("consistent", [False, True])
def test_p5_taylor_green_decay_c1(consistent):
    """C1 (z-invariant 2-D Taylor-Green, omega = 1.8): amplitude ~ exp(-2 nu k^2 t); north_star
    asks 1 %.  Fit from step 20 (zero Pi^neq start) or from 0 with the consistent Pi^neq start."""
    om = 1.8
    d = inputs.taylor_green_2d(32, 0.02, om, consistent_pineq=consistent, nz=2)
    o = ref.Oracle(32, 32, 2, om)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], None, d["pineq"])
    amp = []
    for _ in range(101):
        m = o.get_moments()
        amp.append(((m["ux"] * d["ux"]) + (m["uy"] * d["uy"])).sum() / (d["ux"] ** 2 + d["uy"] ** 2).sum())
        o.step(1)
    nu = CS2 * (1 / om - 0.5)
    k = 2 * math.pi / 32
    s0 = 0 if consistent else 20
    rate = -np.polyfit(np.arange(s0, 101), np.log(np.array(amp[s0:])), 1)[0]
    assert abs(rate / (2 * nu * k * k) - 1) < 2e-3
    assert abs(amp[100] / math.exp(-2 * nu * k * k * 100) - 1) < (2e-3 if consistent else 1e-2)
    assert abs(m["uz"]).max() < 1e-16


# ---------------------------------------------------------------- P6 fixed points / reductions
def test_p6_uniform_equilibrium_is_a_fixed_point():
    shape = (6, 5, 7)
    one = np.ones(shape)
    for phi_c in (0.0, 1.0):
        d = dict(rho=1.02 * one, ux=0.03 * one, uy=-0.02 * one, uz=0.01 * one, phi=phi_c * one)
        o = _run(d, 1.6, 7, sigma=0.02, interface_width=4.0)
        m = o.get_moments()
        np.testing.assert_allclose(m["rho"], 1.02, atol=1e-15)
        np.testing.assert_allclose(m["ux"], 0.03, atol=1e-16)
        np.testing.assert_allclose(m["uy"], -0.02, atol=1e-16)
        np.testing.assert_allclose(m["uz"], 0.01, atol=1e-16)
        np.testing.assert_allclose(m["pineq"], 0, atol=1e-16)
        np.testing.assert_allclose(m["phi"], phi_c, atol=1e-15)


def test_p6_sigma_zero_is_single_component_bit_for_bit():
    """without surface tension the flow half is the single-component TSLB."""
    d = inputs.smooth_random(8, 9, 10, seed=5)
    o2 = _run(d, 1.9, 6, sigma=0.0, interface_width=3.0)
    d1 = dict(d)
    d1["phi"] = None
    o1 = _run(d1, 1.9, 6)
    m2, m1 = o2.get_moments(), o1.get_moments()
    for k in ("rho", "ux", "uy", "uz", "pineq"):
        assert np.array_equal(m1[k], m2[k])


# ---------------------------------------------------------------- P7 phase step, exact factor
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p7_phase_step_amplification_factor(axis):
    """PAPER.md:206 eq. 23 on D3Q7 (w0 = 1/4, w = 1/8, c_sg^2 = 1/4; A8) with gamma -> 0: a
    Fourier mode along an axis with uniform velocity u along it is multiplied per step by exactly
    lambda = 3/4 + cos(k)/4 - i u sin(k)."""
    n = 16
    shape = [4, 4, 4]
    shape[2 - axis] = n                       # arrays are (nz, ny, nx)
    s = np.arange(n).reshape([n if i == 2 - axis else 1 for i in range(3)]) + np.zeros(shape)
    k = 2 * math.pi * 3 / n
    uval = 0.07
    one = np.ones(shape)
    u = [0 * one, 0 * one, 0 * one]
    u[axis] = uval * one
    phi0 = 0.4 + 0.3 * np.cos(k * s)
    d = dict(rho=one, ux=u[0], uy=u[1], uz=u[2], phi=phi0)
    lam = 0.75 + 0.25 * math.cos(k) - 1j * uval * math.sin(k)
    steps = 5
    o = _run(d, 1.3, steps, sigma=0.0, interface_width=1e300)
    # lambda is the factor of e^{+iks}; cos(ks) = Re e^{+iks}
    expect = 0.4 + 0.3 * np.real(lam ** steps * np.exp(1j * k * s))
    got = o.get_moments()["phi"]
    assert np.abs(got - expect).max() < 1e-15
    # a wrong advection sign (lambda conjugated) is resolved by this test
    assert np.abs(got - (0.4 + 0.3 * np.real(np.conj(lam) ** steps * np.exp(1j * k * s)))).max() > 1e-3
    # u = 0: pure diffusion with D = c_sg^2 (1 - 1/2) = 1/8 (small-k limit of 3/4 + cos(k)/4)
    assert abs((1 - (0.75 + 0.25 * math.cos(1e-3))) / 1e-6 - 1 / 8) < 1e-6


# ---------------------------------------------------------------- P8 planar interface
def test_p8_planar_interface_is_stationary():
    """PAPER.md:202, 211 with gamma = 2/W (A8): phi = 1/2 (1 + tanh(2 s / W)) stays put."""
    nz, W = 96, 4.0
    z = np.arange(nz, dtype=float).reshape(nz, 1, 1) + np.zeros((nz, 4, 4))
    phi = 0.5 * (np.tanh(2 * (z - 24) / W) - np.tanh(2 * (z - 72) / W))
    one = np.ones_like(phi)
    d = dict(rho=one, ux=0 * one, uy=0 * one, uz=0 * one, phi=phi)

    def width(p):
        return 1.0 / np.abs((np.roll(p, -1, 0) - np.roll(p, 1, 0)) / 2)[:48].max()

    def level(p):
        col = p[:48, 0, 0]
        j = np.where((col[:-1] < 0.5) & (col[1:] >= 0.5))[0][0]
        return j + (0.5 - col[j]) / (col[j + 1] - col[j])

    w0, l0 = width(phi), level(phi)
    o = _run(d, 1.0, 1000, sigma=0.01, interface_width=W)
    m = o.get_moments()
    assert abs(level(m["phi"]) - l0) < 1e-6
    assert abs(width(m["phi"]) / w0 - 1) < 0.05
    assert max(np.abs(m[k]).max() for k in ("ux", "uy", "uz")) < 1e-10
    assert m["phi"].min() > -1e-6 and m["phi"].max() < 1 + 1e-6
    o.step(500)
    assert abs(width(o.get_moments()["phi"]) / width(m["phi"]) - 1) < 2e-3   # steady


# ---------------------------------------------------------------- P9 Young-Laplace
def _laplace(n, R, W, sigma, steps, navg, omega=1.0):
    d = inputs.static_droplet(n, R, W)
    # pre-load the Laplace pressure to cut box-acoustic ringing (protocol)
    rho = 1 + (2 * sigma / (R * CS2)) * (d["phi"] - d["phi"].mean())
    o = ref.Oracle(n, n, n, omega, two_component=True, sigma=sigma, interface_width=W)
    o.init_fields(rho, d["ux"], d["uy"], d["uz"], d["phi"])
    x, y, z = inputs.grid(n, n, n)
    c = (n - 1) / 2
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    inside, outside = r < R / 2, r > R + (n / 2 - R) / 2
    o.step(steps - navg)
    dps = []
    for _ in range(navg):
        o.step(1)
        m = o.get_moments()
        dps.append(CS2 * (m["rho"][inside].mean() - m["rho"][outside].mean()))
    return float(np.mean(dps)), o


def test_p9_young_laplace_small():
    """PAPER.md:188 ("compliant with the Young-Laplace law"): dp = 2 sigma / R, here R = 8 in 32^3
    with W/R = 1/2 where the finite-width excess is ~ +4 %; fixes the sign and
    normalisation of F = sigma kappa grad(phi) (A6) and the unit weight of the kick (A9)."""
    n, R, W, sigma = 32, 8.0, 4.0, 0.01
    dp, o = _laplace(n, R, W, sigma, steps=411, navg=111)
    ratio = dp / (2 * sigma / R)
    assert 1.0 < ratio < 1.06, ratio
    # mechanical balance against the oracle's own force field along a lattice axis through the
    # droplet: p_in - p_out = - sum F_x dx  (kick adds exactly F: a factor 1/2 or 2 fails this)
    _, _, _, F = o.phase_geometry()
    c = n // 2
    line = -F[0][c, c, c:].sum()
    assert abs(line / dp - 1) < 0.03, (line, dp)
    # linear in sigma
    dp2, _ = _laplace(n, R, W, sigma / 4, steps=411, navg=111)
    assert abs(dp2 * 4 / dp - 1) < 0.01


@pytest.mark.slow
def test_p9_young_laplace_c2_full():
    """C2 exactly: 64^3, R = 16, W = 4, sigma = 0.01, omega = 1, 2000 steps, average over the last
    2 nx / c_s steps.  ~7 min on 8 cores; the value is also stored in tests/golden/."""
    dp, _ = _laplace(64, 16.0, 4.0, 0.01, steps=2000, navg=222)
    assert abs(dp / (2 * 0.01 / 16.0) - 1) < 0.02


# ---------------------------------------------------------------- P10 brute force 8^3
@pytest.mark.parametrize("order", [3, 2])
def test_p10_brute_force_8cubed(order):
    d = inputs.smooth_random(8, 8, 8, seed=11)
    omega, sigma, W = 1.85, 0.02, 3.0
    o = ref.Oracle(8, 8, 8, omega, two_component=True, sigma=sigma, interface_width=W,
                   hermite_order=order)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"], d["pineq"])
    b = BruteForce(omega, sigma, W, two=True, order=order)
    b.init(d["rho"], np.stack([d["ux"], d["uy"], d["uz"]]), d["phi"], d["pineq"])
    # populations agree right after init (as sets: the two orderings differ)
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
    assert np.abs(b.pineq6).max() > 1e-4 and np.abs(b.u).max() > 1e-3


# ---------------------------------------------------------------- P11 equivariance
def _transform(d, perm, flips, shift):
    """Apply a lattice symmetry (axis permutation + reflections) and a periodic translation to a
    state dict.  perm maps new spatial axis a -> old axis perm[a] (axes x=0,y=1,z=2)."""
    def sc(a):            # scalar field, array axes are (z, y, x) = spatial (2, 1, 0)
        arr_axes = [2 - perm[2 - i] for i in range(3)]
        b = np.transpose(a, arr_axes)
        for ax in range(3):
            if flips[ax]:
                b = np.flip(b, axis=2 - ax)
        return np.roll(b, shift=(shift[2], shift[1], shift[0]), axis=(0, 1, 2))

    sgn = [(-1.0 if f else 1.0) for f in flips]
    u_old = [d["ux"], d["uy"], d["uz"]]
    out = dict(rho=sc(d["rho"]), phi=None if d.get("phi") is None else sc(d["phi"]))
    unew = [sgn[a] * sc(u_old[perm[a]]) for a in range(3)]
    out["ux"], out["uy"], out["uz"] = unew
    if d.get("pineq") is not None:
        P = {(0, 0): 0, (1, 1): 1, (2, 2): 2, (0, 1): 3, (1, 0): 3, (0, 2): 4, (2, 0): 4, (1, 2): 5, (2, 1): 5}
        pn = [None] * 6
        for (a, b), k in P.items():
            pn[k] = sgn[a] * sgn[b] * sc(d["pineq"][P[(perm[a], perm[b])]])
        out["pineq"] = np.stack(pn)
    else:
        out["pineq"] = None
    return out


@pytest.mark.parametrize("perm,flips,shift", [
    ((1, 0, 2), (False, False, False), (0, 0, 0)),
    ((2, 0, 1), (True, False, False), (1, 2, 3)),
    ((0, 2, 1), (False, True, True), (3, 0, 5)),
    ((2, 1, 0), (True, True, True), (0, 4, 0)),
    ((0, 1, 2), (False, False, True), (2, 2, 2)),
])
def test_p11_lattice_equivariance(perm, flips, shift):
    d = inputs.smooth_random(8, 8, 8, seed=21)
    kw = dict(sigma=0.015, interface_width=3.0)
    steps = 3
    o = _run(d, 1.8, steps, **kw)
    m = o.get_moments()
    m_t = _transform(m, perm, flips, shift)
    o2 = _run(_transform(d, perm, flips, shift), 1.8, steps, **kw)
    m2 = o2.get_moments()
    for k in ("rho", "ux", "uy", "uz", "phi", "pineq"):
        scale = max(np.abs(m2[k]).max(), 1e-30)
        assert np.abs(m2[k] - m_t[k]).max() / scale < 1e-11, k


# ---------------------------------------------------------------- P12 stencils
def test_p12_gradient_stencil_fourier_symbol_and_curvature():
    """A7: G_a = central difference along a, smoothed by [1/6, 2/3, 1/6] along the other two axes
    (the D3Q27 isotropic gradient).  Its exact Fourier symbol on a plane wave is
    i sin(k_a) (2 + cos k_b)/3 (2 + cos k_g)/3; kappa of a sphere is 2/r."""
    n = 12
    x, y, z = inputs.grid(n, n, n)
    kx, ky, kz = 2 * math.pi / n * np.array([1, 2, 3])
    ph = kx * x + ky * y + kz * z + 0.3
    one = np.ones_like(x)
    d = dict(rho=one, ux=0 * one, uy=0 * one, uz=0 * one, phi=0.5 + 0.2 * np.sin(ph))
    o = _run(d, 1.0, 0, sigma=0.01, interface_width=4.0)
    G, nn, kappa, F = o.phase_geometry()
    sm = lambda k: (2 + math.cos(k)) / 3
    np.testing.assert_allclose(G[0], 0.2 * math.sin(kx) * sm(ky) * sm(kz) * np.cos(ph), atol=1e-15)
    np.testing.assert_allclose(G[1], 0.2 * sm(kx) * math.sin(ky) * sm(kz) * np.cos(ph), atol=1e-15)
    np.testing.assert_allclose(G[2], 0.2 * sm(kx) * sm(ky) * math.sin(kz) * np.cos(ph), atol=1e-15)
    np.testing.assert_allclose((nn * nn).sum(0), 1.0, atol=1e-9)
    np.testing.assert_allclose(F, 0.01 * kappa[None] * G, atol=1e-18)
    # curvature of a sphere, R = 12 in 40^3: kappa ~ 2/r in the interface shell, sign + (A6)
    n, R = 40, 12.0
    d = inputs.static_droplet(n, R, 4.0)
    o = _run(d, 1.0, 0, sigma=0.01, interface_width=4.0)
    G, nn, kappa, F = o.phase_geometry()
    x, y, z = inputs.grid(n, n, n)
    c = (n - 1) / 2
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    shell = np.abs(r - R) < 2.0
    assert np.abs(kappa[shell] * r[shell] / 2 - 1).max() < 0.05
    # n points along grad(phi): inward for a phi = 1 droplet
    nr = (nn[0] * (x - c) + nn[1] * (y - c) + nn[2] * (z - c)) / r
    assert nr[shell].max() < -0.999


# ---------------------------------------------------------------- jet boundaries (A10/A11: parity unpinned)
def test_jet_boundary_planes_sanity():
    """Inflow/outflow (eqs. 9-10 as read in A10/A11): imposed values are what is
    stored, one-step memory of the neighbour plane, fields stay bounded.  (The rebuilt populations and the
    mass / momentum fluxes through the two planes: test_jet_boundary_populations_are_eq9,
    test_jet_mass_balance_from_boundary_populations.)"""
    nx, ny, nz, D, U, pert, seed = 24, 24, 40, 8.0, 0.05, 0.05, 2024
    prm = inputs.jet_params(nx, ny, nz, D, U=U, Re=500.0, We=200.0, perturbation=pert, seed=seed)
    d = inputs.jet_quiescent(nx, ny, nz)
    o = ref.Oracle(nx, ny, nz, prm["omega"], two_component=True, sigma=prm["sigma"],
                   interface_width=4.0, bc_zlo=ref.BC_JET_INFLOW, bc_zhi=ref.BC_OUTFLOW,
                   jet_diameter=D, jet_velocity=U, jet_perturbation=pert, seed=seed)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    x, y, _ = inputs.grid(nx, ny, 1)
    disc = ((x[0] - (nx - 1) / 2) ** 2 + (y[0] - (ny - 1) / 2) ** 2) < (D / 2) ** 2
    for step in (0, 1, 2, 60):
        if step:
            prev = o.get_moments()
            o.step(step - o_step)
        o_step = step
        m = o.get_moments()
        xi = np.array([[ref.xi(seed, i, j, nx, ny, step) for i in range(nx)] for j in range(ny)])
        np.testing.assert_allclose(m["uz"][0], np.where(disc, U * (1 + pert * xi), 0.0), atol=1e-18)
        assert np.all(m["ux"][0] == 0) and np.all(m["uy"][0] == 0)
        assert np.array_equal(m["phi"][0], disc.astype(float))
        assert np.all(m["rho"][-1] == 1.0)
        if step in (1, 2):      # one-step memory of the neighbour plane (A11: OLD values)
            assert np.array_equal(m["rho"][0], prev["rho"][1])
            assert np.array_equal(m["pineq"][:, 0], prev["pineq"][:, 1])
            assert np.array_equal(m["uz"][-1], prev["uz"][-2])
            assert np.array_equal(m["phi"][-1], prev["phi"][-2])
    assert disc.sum() == 52
    assert -1e-3 < m["phi"].min() and m["phi"].max() < 1 + 1e-3
    assert 0.97 < m["rho"].min() and m["rho"].max() < 1.03
    assert m["phi"][1:6].sum() > 100           # fluid A has entered
    assert np.isfinite(m["pineq"]).all()


def _jet_oracle(nx, ny, nz, D, forcing=None, steps=0, seed=2024, pert=0.05, U=0.05):
    prm = inputs.jet_params(nx, ny, nz, D, U=U, Re=300.0, We=20.0, perturbation=pert, seed=seed)
    d = inputs.jet_developed(nx, ny, nz, D, U=U, ndrop=3)
    rng = np.random.default_rng(11)
    for k in ("ux", "uy"):      # transverse motion, so that Pi^neq and u differ from plane to plane
        d[k] = 0.01 * rng.standard_normal(d[k].shape)
    kw = {} if forcing is None else dict(forcing=forcing)
    o = ref.Oracle(nx, ny, nz, prm["omega"], two_component=True, sigma=prm["sigma"], interface_width=4.0,
                   bc_zlo=ref.BC_JET_INFLOW, bc_zhi=ref.BC_OUTFLOW, jet_diameter=D, jet_velocity=U,
                   jet_perturbation=pert, seed=seed, **kw)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    if steps:
        o.step(steps)
    return o, prm


def test_jet_boundary_populations_are_eq9():
    """PAPER.md:125-137 eqs. 9-10: f_i(x_B) = f_i^eq(rho_B, u_B) + (1 - omega) f_i^neq(Pi^neq(x_F), u_B) with the
    IMPOSED rho_B, u_B of reading A10 and the neighbour plane's Pi^neq.  The populations the oracle holds
    on the two boundary planes are compared with that formula rebuilt from the probes ref.feq / ref.fneq
    (pinned by P2, P3).  A missing (1 - omega), a velocity taken from x_F, or a forgotten rebuild fails."""
    nx, ny, nz, D = 20, 18, 16, 8.0
    o, prm = _jet_oracle(nx, ny, nz, D, steps=3)
    prev = o.get_moments()
    o.step(1)
    m = o.get_moments()
    f = o.get_populations()
    omc = 1.0 - prm["omega"]
    assert abs(omc) > 0.3
    worst = 0.0
    for zb, zf in ((0, 1), (nz - 1, nz - 2)):
        # the stored Pi^neq of the boundary plane is the OLD one of the fluid neighbour (A11), and it is not small
        assert np.array_equal(m["pineq"][:, zb], prev["pineq"][:, zf])
        assert np.abs(m["pineq"][:, zb]).max() > 1e-6
        # the imposed velocity differs from the neighbour's
        assert np.abs(m["uz"][zb] - m["uz"][zf]).max() > 1e-4
        for y in range(ny):
            for x in range(nx):
                u = np.array([m["ux"][zb, y, x], m["uy"][zb, y, x], m["uz"][zb, y, x]])
                want = ref.feq(m["rho"][zb, y, x], u) + omc * ref.fneq(m["pineq"][:, zb, y, x], u)
                worst = max(worst, np.abs(f[:, zb, y, x] - want).max())
    assert worst < 1e-15, worst
    o.close()


def test_jet_mass_balance_from_boundary_populations():
    """Reading A10, its pin: the interior mass changes per step by exactly what the boundary-plane
    populations carry in minus what the interior sends to the two planes, and the net inlet mass flux is
    sum_nozzle rho_B U (1 + p xi)  (first moment of the rebuilt inlet populations = the imposed momentum)."""
    nx, ny, nz, D, U, pert, seed = 20, 18, 16, 8.0, 0.05, 0.05, 2024
    o, prm = _jet_oracle(nx, ny, nz, D, steps=2, U=U, pert=pert, seed=seed)
    c, w = ref.lattice()
    up, dn = c[:, 2] == 1, c[:, 2] == -1
    x, y, _ = inputs.grid(nx, ny, 1)
    disc = ((x[0] - (nx - 1) / 2) ** 2 + (y[0] - (ny - 1) / 2) ** 2) < (D / 2) ** 2
    for t in (2, 3, 4):
        m0 = o.get_moments()
        f = o.get_populations()                       # post-collision populations of time t
        assert abs(f[:, 1:-1].sum() - m0["rho"][1:-1].sum()) < 1e-10   # collision keeps the mass
        o.step(1)
        m1 = o.get_moments()
        gain = f[up, 0].sum() + f[dn, nz - 1].sum()       # from the two boundary planes into planes 1 and nz-2
        loss = f[dn, 1].sum() + f[up, nz - 2].sum()       # from planes 1 and nz-2 into the boundary planes
        dm = m1["rho"][1:-1].sum() - m0["rho"][1:-1].sum()
        assert abs(dm - (gain - loss)) < 1e-11 * max(gain, 1.0), (t, dm, gain - loss)
        # net inlet flux = first z-moment of the inlet populations = imposed rho_B u_B
        xi = np.array([[ref.xi(seed, i, j, nx, ny, t) for i in range(nx)] for j in range(ny)])
        flux = (f[:, 0] * c[:, 2][:, None, None]).sum()
        want = (m0["rho"][0] * np.where(disc, U * (1 + pert * xi), 0.0)).sum()
        assert abs(flux - want) < 1e-13, (t, flux, want)
        assert want > 0.5 * disc.sum() * U
        # and no transverse momentum comes in
        assert abs((f[:, 0] * c[:, 0][:, None, None]).sum()) < 1e-14
    o.close()


def test_guo_jet_momentum_balance_with_unforced_boundary_planes():
    """Reading A18 with inflow/outflow: F = 0 on the two imposed planes.  (i) the first moment of the
    boundary-plane populations is exactly the imposed rho_B u_B although grad(phi) is not zero there (nozzle
    rim); (ii) the bare interior momentum obeys  sum m(t+1) = sum (m(t) + F(t)) + (what the boundary
    populations carry in) - (what the interior sends out),  F = sigma kappa grad(phi) of the time-t phi."""
    nx, ny, nz, D = 20, 18, 16, 8.0
    o, prm = _jet_oracle(nx, ny, nz, D, forcing=ref.FORCING_GUO, steps=2)
    c, w = ref.lattice()
    up, dn = c[:, 2] == 1, c[:, 2] == -1
    for t in (2, 3):
        m0 = o.get_moments()
        G, nn, kappa, F = o.phase_geometry()
        assert np.abs(G[:, 0]).max() > 1e-3                # the nozzle rim: a force would be there
        f = o.get_populations()
        for zb in (0, nz - 1):
            for a, key in enumerate(("ux", "uy", "uz")):
                mom = (f[:, zb] * c[:, a][:, None, None]).sum(axis=0)
                assert np.abs(mom - m0["rho"][zb] * m0[key][zb]).max() < 1e-16
        o.step(1)
        m1 = o.get_moments()
        for a, key in enumerate(("ux", "uy", "uz")):
            ca = c[:, a][:, None, None]
            gain = (f[up, 0] * ca[up]).sum() + (f[dn, nz - 1] * ca[dn]).sum()
            loss = (f[dn, 1] * ca[dn]).sum() + (f[up, nz - 2] * ca[up]).sum()
            before = (m0["rho"][1:-1] * m0[key][1:-1]).sum() + F[a, 1:-1].sum()
            after = (m1["rho"][1:-1] * m1[key][1:-1]).sum()
            assert abs(after - (before + gain - loss)) < 1e-12, (t, key, after - (before + gain - loss))
        assert np.abs(F[:, 1:-1]).max() > 1e-7
    o.close()

"""Seeded synthetic input generators (numpy only).

This module holds NONE of the method's arithmetic: it only builds initial fields and parameter
sets with the shapes, value ranges and structure of the paper's workloads as
restated in BASELINE.json configs C1..C5 (recipe: DESIGN.md §4).  Both the CPU oracle and the
CUDA library are fed from here; neither imports the other.

All fields are float64 arrays of shape (nz, ny, nx), x fastest.
"""
import math

import numpy as np

CS2 = 1.0 / 3.0


def omega_from_nu(nu):
    """nu = c_s^2 (1/omega - 1/2)."""
    return 1.0 / (nu / CS2 + 0.5)


def grid(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                          np.arange(nx, dtype=np.float64), indexing="ij")
    return x, y, z


def taylor_green_2d(n=32, U0=0.02, omega=1.8, consistent_pineq=False, nz=None):
    """C1: z-invariant 2-D Taylor-Green vortex (an exact Navier-Stokes solution, decays as
    exp(-2 nu k^2 t)).  Returns dict(rho, ux, uy, uz, pineq or None)."""
    nz = n if nz is None else nz
    x, y, _ = grid(n, n, nz)
    k = 2.0 * math.pi / n
    ux = -U0 * np.cos(k * x) * np.sin(k * y)
    uy = U0 * np.sin(k * x) * np.cos(k * y)
    uz = np.zeros_like(ux)
    rho = 1.0 - (3.0 * U0 * U0 / 4.0) * (np.cos(2 * k * x) + np.cos(2 * k * y))
    pin = None
    if consistent_pineq:
        # Pi^neq = -(rho c_s^2 / omega)(d_a u_b + d_b u_a), analytic derivatives
        dxux = U0 * k * np.sin(k * x) * np.sin(k * y)
        dyuy = -U0 * k * np.sin(k * x) * np.sin(k * y)
        dyux = -U0 * k * np.cos(k * x) * np.cos(k * y)
        dxuy = U0 * k * np.cos(k * x) * np.cos(k * y)
        f = -rho * CS2 / omega
        zero = np.zeros_like(ux)
        pin = np.stack([f * 2 * dxux, f * 2 * dyuy, zero, f * (dyux + dxuy), zero, zero])
    return dict(rho=rho, ux=ux, uy=uy, uz=uz, pineq=pin, phi=None)


def taylor_green_3d(n=32, U0=0.02):
    """C1 extra (parity only): classic 3-D TGV initial field."""
    x, y, z = grid(n, n, n)
    k = 2.0 * math.pi / n
    ux = U0 * np.sin(k * x) * np.cos(k * y) * np.cos(k * z)
    uy = -U0 * np.cos(k * x) * np.sin(k * y) * np.cos(k * z)
    uz = np.zeros_like(ux)
    rho = 1.0 + (3.0 * U0 * U0 / 16.0) * (np.cos(2 * k * x) + np.cos(2 * k * y)) * (np.cos(2 * k * z) + 2.0)
    return dict(rho=rho, ux=ux, uy=uy, uz=uz, pineq=None, phi=None)


def shear_wave(nx, ny, nz, U0=0.01, axis="y"):
    """u_x = U0 sin(k y) (or k z): decays as exp(-nu k^2 t)."""
    x, y, z = grid(nx, ny, nz)
    if axis == "y":
        ux = U0 * np.sin(2.0 * math.pi / ny * y)
    else:
        ux = U0 * np.sin(2.0 * math.pi / nz * z)
    zero = np.zeros_like(ux)
    return dict(rho=np.ones_like(ux), ux=ux, uy=zero.copy(), uz=zero.copy(), pineq=None, phi=None)


def static_droplet(n=64, R=16.0, W=4.0):
    """C2: phi = 1/2 (1 - tanh(2 (r - R)/W)) centred at ((n-1)/2)^3, rho = 1, u = 0."""
    x, y, z = grid(n, n, n)
    c = (n - 1) / 2.0
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    phi = 0.5 * (1.0 - np.tanh(2.0 * (r - R) / W))
    one = np.ones_like(phi)
    zero = np.zeros_like(phi)
    return dict(rho=one, ux=zero, uy=zero.copy(), uz=zero.copy(), pineq=None, phi=phi)


def droplets_noise(nx, ny=None, nz=None, seed=12345, ndrop=40, rmin=6.0, rmax=12.0, W=4.0,
                   noise=0.01):
    """C3: seeded spherical inclusions (periodic minimum-image distance) plus iid uniform velocity
    noise in [-noise, noise]; rho = 1."""
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    rng = np.random.default_rng(seed)
    cx = rng.uniform(0, nx, ndrop)
    cy = rng.uniform(0, ny, ndrop)
    cz = rng.uniform(0, nz, ndrop)
    rad = rng.uniform(rmin, rmax, ndrop)
    x1 = np.arange(nx, dtype=np.float64)
    y1 = np.arange(ny, dtype=np.float64)
    z1 = np.arange(nz, dtype=np.float64)
    phi = np.zeros((nz, ny, nx))
    for k in range(ndrop):
        dx = np.abs(x1 - cx[k]); dx = np.minimum(dx, nx - dx)
        dy = np.abs(y1 - cy[k]); dy = np.minimum(dy, ny - dy)
        dz = np.abs(z1 - cz[k]); dz = np.minimum(dz, nz - dz)
        d = np.sqrt(dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2)
        np.maximum(phi, 0.5 * (1.0 - np.tanh(2.0 * (d - rad[k]) / W)), out=phi)
    ux = rng.uniform(-noise, noise, phi.shape)
    uy = rng.uniform(-noise, noise, phi.shape)
    uz = rng.uniform(-noise, noise, phi.shape)
    return dict(rho=np.ones_like(phi), ux=ux, uy=uy, uz=uz, pineq=None, phi=phi)


def smooth_random(nx, ny, nz, seed=7, amp_u=0.02, amp_rho=0.01, amp_pi=1e-3, blob=True):
    """Small smooth random fields (a few low Fourier modes per field) with a phi blob; used by
    the brute-force and equivariance pins."""
    rng = np.random.default_rng(seed)
    x, y, z = grid(nx, ny, nz)

    def modes(amp):
        f = np.zeros((nz, ny, nx))
        for _ in range(4):
            kx, ky, kz = rng.integers(0, 3, 3)
            ph = rng.uniform(0, 2 * math.pi)
            f += rng.uniform(-1, 1) * np.cos(2 * math.pi * (kx * x / nx + ky * y / ny + kz * z / nz) + ph)
        return amp * f / 4.0

    d = dict(rho=1.0 + modes(amp_rho), ux=modes(amp_u), uy=modes(amp_u), uz=modes(amp_u))
    d["pineq"] = np.stack([modes(amp_pi) for _ in range(6)])
    if blob:
        cx, cy, cz = (nx - 1) / 2.0 + 0.3, (ny - 1) / 2.0 - 0.2, (nz - 1) / 2.0 + 0.1
        r = np.sqrt((x - cx) ** 2 + (y - cy) ** 2 + (z - cz) ** 2)
        d["phi"] = 0.5 * (1.0 - np.tanh(2.0 * (r - min(nx, ny, nz) / 4.0) / 3.0))
    else:
        d["phi"] = None
    return d


def jet_params(nx, ny, nz, D, U=0.05, Re=5000.0, We=2000.0, perturbation=0.05, seed=2024, W=4.0):
    """C4/C5 parameter set: nu = U D / Re, sigma = rho U^2 D / We (BASELINE.json; A14)."""
    nu = U * D / Re
    return dict(nx=nx, ny=ny, nz=nz, omega=omega_from_nu(nu), sigma=U * U * D / We,
                interface_width=W, two_component=True, jet=True, jet_diameter=float(D),
                jet_velocity=U, jet_perturbation=perturbation, seed=seed)


def jet_quiescent(nx, ny, nz):
    """C4/C5 initial state: rho = 1, u = 0, phi = 0 (the inlet plane is set by the library)."""
    one = np.ones((nz, ny, nx))
    zero = np.zeros((nz, ny, nx))
    return dict(rho=one, ux=zero, uy=zero.copy(), uz=zero.copy(), pineq=None, phi=zero.copy())


def jet_developed(nx, ny, nz, D, U=0.05, seed=99, ndrop=200, W=4.0):
    """Optional 'developed' jet-shaped state (throughput is data independent; this shows it):
    a phi core of diameter D over the first third of z, seeded droplets in a cone downstream and
    an axial velocity with the self-similar profile shape exp(-75 (r/(z+z0))^2) of PAPER.md:271."""
    rng = np.random.default_rng(seed)
    x1 = np.arange(nx) - (nx - 1) / 2.0
    y1 = np.arange(ny) - (ny - 1) / 2.0
    z1 = np.arange(nz, dtype=np.float64)
    r = np.sqrt(y1[None, :, None] ** 2 + x1[None, None, :] ** 2) + 0.0 * z1[:, None, None]
    zz = z1[:, None, None] + 0.0 * r
    z0 = 6.0 * D
    uz = U * np.exp(-75.0 * (r / (zz + z0)) ** 2)
    core = 0.5 * (1.0 - np.tanh(2.0 * (r - D / 2.0) / W)) * (zz < nz / 3.0)
    phi = core
    for _ in range(ndrop):
        cz = rng.uniform(nz / 3.0, max(nz / 3.0 + 1.0, nz - 8.0))
        spread = 0.1 * (cz + z0)
        cx, cy = rng.normal(0, spread, 2)
        rad = rng.uniform(3.0, 0.2 * D + 3.0)
        lo, hi = int(max(cz - rad - 6, 0)), int(min(cz + rad + 7, nz))
        d = np.sqrt((z1[lo:hi, None, None] - cz) ** 2 + (y1[None, :, None] - cy) ** 2 +
                    (x1[None, None, :] - cx) ** 2)
        phi[lo:hi] = np.maximum(phi[lo:hi], 0.5 * (1.0 - np.tanh(2.0 * (d - rad) / W)))
    zero = np.zeros_like(phi)
    return dict(rho=np.ones_like(phi), ux=zero, uy=zero.copy(), uz=uz, pineq=None, phi=phi)

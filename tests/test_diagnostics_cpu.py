"""Host post-processing (paper_2403_15773_b200/diagnostics.py) on synthetic averages with known
answers: a self-similar jet  <u_z>(r, z) = U B D/(z - z0) exp(-K (r/(z - z0))^2)  (the form the paper
fits) must give back its centre-line slope 1/(B D) and its exponent K.  CPU only."""
import numpy as np

from paper_2403_15773_b200 import diagnostics


def test_centerline_fit_and_gaussian_exponent_of_a_synthetic_self_similar_jet():
    nx, nz, D, U, B, K, z0 = 400, 800, 40.0, 0.05, 6.5, 75.0, -30.0
    x = np.arange(nx) - (nx - 1) / 2.0
    z = np.arange(nz, dtype=np.float64)
    zz = np.maximum(z - z0, 1.0)[:, None]
    avg = U * B * D / zz * np.exp(-K * (x[None, :] / zz) ** 2)
    c = diagnostics.centerline(avg)
    # the two middle columns sit at r = 1/2: centre-line value up to exp(-K/(4 zeff^2))
    assert np.allclose(c[200:] * (z[200:] - z0) / (U * B * D), 1.0, atol=1e-3)
    inv = diagnostics.inverse_centerline(avg, scale=U)
    zD = z / D
    sel = (zD >= 8) & (zD <= 16)
    slope, icpt, rms = diagnostics.linear_fit(zD[sel], inv[sel])
    assert abs(slope * B - 1) < 1e-3 and rms < 1e-4
    assert abs(-icpt / slope * D - z0) < 0.5                    # virtual origin
    r, q = diagnostics.radial_profile(avg, 480)
    assert np.all(np.diff(r) >= 0) and r[0] == 0.5
    Kfit = diagnostics.gaussian_exponent(r, q, 480 - z0)
    assert abs(Kfit / K - 1) < 0.02
    assert diagnostics.gaussian_exponent(r, 0 * q, 480 - z0) is None

"""Host post-processing of the mid-plane time averages returned by Tslb.stats_get()
(Figs. 5-6): centre-line values and radial profiles.  numpy only; the averages
themselves are accumulated on the GPU (tslb_stats_begin / tslb_stats_get)."""
import numpy as np


def centerline(avg):
    """avg: (nz, nx) time average on the mid x-z plane -> its value on the jet axis x = (nx-1)/2 for
    every z (mean of the two middle columns when nx is even)."""
    nx = avg.shape[1]
    return 0.5 * (avg[:, (nx - 1) // 2] + avg[:, nx // 2])


def inverse_centerline(avg, scale=1.0):
    """scale / <q_c>(z): the quantity whose growth beyond the potential core the paper fits with a
    straight line of slope ~ 1/(6.5 D)."""
    c = centerline(avg)
    return scale / np.where(np.abs(c) > 1e-300, c, np.nan)


def radial_profile(avg, z):
    """-> (r, q): distance from the axis and the time average at height z, both sides folded."""
    nx = avg.shape[1]
    r = np.abs(np.arange(nx) - (nx - 1) / 2.0)
    order = np.argsort(r, kind="stable")
    return r[order], avg[z][order]


def linear_fit(x, y):
    """Least-squares line y = slope * x + intercept -> (slope, intercept, rms residual)."""
    a = np.vstack([x, np.ones_like(x)]).T
    (slope, icpt), _, _, _ = np.linalg.lstsq(a, y, rcond=None)
    r = y - (slope * x + icpt)
    return float(slope), float(icpt), float(np.sqrt((r ** 2).mean()))


def gaussian_exponent(r, q, zeff, lo=0.1, hi=0.95):
    """K of the best fit q(r)/q_c = exp(-K (r/zeff)^2) (K = 75 for <u_z> at 12 D with
    zeff = z - z0), least squares on ln(q/q_c) over the points with lo < q/q_c < hi; r sorted
    ascending (radial_profile), q_c = mean of the two points next to the axis.  None if too few."""
    qc = q[:2].mean()
    if not qc > 0:
        return None
    ok = (q > lo * qc) & (q < hi * qc)
    if ok.sum() < 5:
        return None
    eta2 = (r[ok] / zeff) ** 2
    return -float(np.sum(np.log(q[ok] / qc) * eta2) / np.sum(eta2 ** 2))

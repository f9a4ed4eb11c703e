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

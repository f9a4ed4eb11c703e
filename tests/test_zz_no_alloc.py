"""tslb_get_physical_velocity_noalloc (include/tslb.h): the entry point for callers that must not allocate.
Its scratch is one file-scope device array of 12 MiB, shared by every call; the test checks its output
against the existing path (tslb_get_physical_velocity, which allocates its scratch) on two calls in a
row -- the second one finds the first one's contents in the array -- in both precisions and forcing
readings, and that a grid beyond the array is refused.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

from paper_2403_15773_b200 import inputs, tslb
from tests.test_parity_gpu import round_inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", [tslb.F32, tslb.F64])
@pytest.mark.parametrize("forcing,kernel", [(tslb.FORCING_KICK, tslb.KERNEL_TILED), (tslb.FORCING_KICK, tslb.KERNEL_GENERIC),
                                            (tslb.FORCING_GUO, tslb.KERNEL_AUTO)])
def test_noalloc_matches_the_allocating_path_twice(precision, forcing, kernel):
    import torch
    d = round_inputs(inputs.droplets_noise(32, 32, 16, seed=9, ndrop=3, rmin=4.0, rmax=6.0, W=4.0, noise=0.01), precision)
    g = tslb.Tslb(32, 32, 16, 1.6, precision=precision, two_component=True, sigma=0.02, kernel=kernel, forcing=forcing)
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    # a second context on the same device shares the scratch array: its call in between must not matter
    d2 = round_inputs(inputs.droplets_noise(32, 32, 16, seed=4, ndrop=2, rmin=3.0, rmax=5.0, W=4.0, noise=0.02), precision)
    g2 = tslb.Tslb(32, 32, 16, 1.9, precision=precision, two_component=True, sigma=0.01, kernel=kernel, forcing=forcing)
    g2.init_fields(d2["rho"], d2["ux"], d2["uy"], d2["uz"], d2["phi"])
    g2.step(2)
    out = torch.full((3, 16, 32, 32), float("nan"), dtype=g.torch_dtype, device=g.device)
    for call in range(2):
        g.step(3)
        want = g.get_physical_velocity(device=True)           # existing path (synchronises the stream)
        g2.get_physical_velocity_noalloc(torch.empty_like(out))   # leaves ITS normals in the shared array
        torch.cuda.synchronize()
        out.fill_(float("nan"))
        g.get_physical_velocity_noalloc(out)
        torch.cuda.synchronize()
        # same kernels, same inputs, same arithmetic: the two paths agree exactly (tolerance of the parity
        # tests, 1e-5 fp32 / 1e-12 fp64, written out for the record)
        tol = 1e-5 if precision == tslb.F32 else 1e-12
        w, o = want.cpu().numpy().astype(np.float64), out.cpu().numpy().astype(np.float64)
        assert np.isfinite(o).all()
        assert np.abs(o - w).max() <= tol * max(np.abs(w).max(), 1e-300), (call, np.abs(o - w).max())
        assert np.array_equal(o, w), call
        assert np.abs(w[0] - g.get_moments()["ux"]).max() > 0      # the force term is really there
    g.close()
    g2.close()


def test_noalloc_refuses_a_grid_beyond_its_array():
    import torch
    lim = tslb.lib().tslb_noalloc_scratch_bytes()
    assert lim == 12 << 20
    g = tslb.Tslb(128, 128, 64, 1.5, precision=tslb.F64, two_component=True, sigma=0.01)   # 3 x 9.7 MB of normals
    d = inputs.droplets_noise(128, 128, 64, seed=1, ndrop=2, rmin=6.0, rmax=9.0, W=4.0, noise=0.0)
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    out = torch.empty((3, 64, 128, 128), dtype=g.torch_dtype, device=g.device)
    with pytest.raises(tslb.TslbError, match="scratch"):
        g.get_physical_velocity_noalloc(out)
    g.get_physical_velocity(device=True)                            # the allocating path still serves it
    g.close()

"""Time averages on the mid x-z plane (include/tslb.h tslb_stats_*; Figs. 5-6)
against the plain definition evaluated on the oracle: <q>(x,z) = (1/N) sum over the sampled steps
of q(x, y_mid, z, t), y_mid = the mean of the two middle rows when ny is even."""
import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import diagnostics, inputs, tslb
from tests.test_parity_gpu import gpu_kwargs, oracle_kwargs, round_inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision,tol", [(tslb.F64, 1e-12), (tslb.F32, 1e-5)])
@pytest.mark.parametrize("shape,every", [((64, 32, 24), 1), ((64, 17, 20), 3)])
def test_midplane_time_averages_match_the_oracle(precision, tol, shape, every):
    nx, ny, nz = shape
    steps = 12
    prm = inputs.jet_params(nx, ny, nz, D=9, U=0.04, Re=300.0, We=50.0, perturbation=0.1, seed=5)
    d = round_inputs(inputs.jet_developed(nx, ny, nz, D=9, ndrop=5), precision)
    g = tslb.Tslb(nx, ny, nz, prm["omega"], precision=precision, **gpu_kwargs(prm))
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    g.step(2)                                   # sampling starts later than the run
    g.stats_begin(every)
    l0 = g.launch_count
    g.step(steps)
    st = g.stats_get()
    assert st["nsamples"] == len([t for t in range(3, 3 + steps) if t % every == 0])
    assert g.launch_count - l0 == 2 * steps + st["nsamples"]      # step + boundary kernel, + one per sample
    o = ref.Oracle(nx, ny, nz, prm["omega"], **oracle_kwargs(prm))
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    o.step(2)
    sp, su, n = np.zeros((nz, nx)), np.zeros((nz, nx)), 0
    ya, yb = (ny - 1) // 2, ny // 2
    for t in range(3, 3 + steps):
        o.step(1)
        if t % every:
            continue
        m = o.get_moments()
        sp += 0.5 * (m["phi"][:, ya, :] + m["phi"][:, yb, :])
        su += 0.5 * (m["uz"][:, ya, :] + m["uz"][:, yb, :])
        n += 1
    o.close()
    assert n == st["nsamples"]
    for got, want in ((st["phi"], sp / n), (st["uz"], su / n)):
        assert np.abs(got - want).max() <= tol * np.abs(want).max()
    # centre-line diagnostics: phi_c = 1 inside the nozzle core near the inlet
    c = diagnostics.centerline(st["phi"])
    assert c.shape == (nz,) and abs(c[0] - 1.0) < 1e-6
    inv = diagnostics.inverse_centerline(st["uz"], scale=prm["jet_velocity"])
    assert np.isfinite(inv[0]) and 0.5 < inv[0] < 2.0
    r, q = diagnostics.radial_profile(st["phi"], 1)
    assert r[0] <= 0.5 and q[0] > 0.9 and q[-1] < 0.1
    # restart and stop
    g.stats_begin(1)
    assert g.stats_get()["nsamples"] == 0
    g.stats_end()
    g.step(1)
    assert g.stats_get()["nsamples"] == 0
    g.close()


def test_stats_single_component_and_errors():
    g = tslb.Tslb(32, 8, 6, 1.2)
    z = np.zeros((6, 8, 32), dtype=np.float32)
    with pytest.raises(tslb.TslbError):
        g.stats_get()
    with pytest.raises(tslb.TslbError):
        g.stats_begin(0)
    g.init_fields(z + 1, z, z, z + 0.01)
    g.stats_begin(2)
    g.step(4)
    st = g.stats_get()
    assert st["phi"] is None and st["nsamples"] == 2
    assert np.allclose(st["uz"], 0.01, rtol=1e-5)
    g.close()

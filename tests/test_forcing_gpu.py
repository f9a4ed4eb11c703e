"""GPU parity of the second forcing reading (TSLB_FORCING_GUO, A18) and of
tslb_get_physical_velocity in both readings, through the C-ABI against the CPU oracle on the same
seeded inputs.  Gates as in test_parity_gpu.py: fp64 1e-12 after 100 steps, fp32 1e-5 after 10."""
import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import inputs, tslb
from tests.test_parity_gpu import TOL, errs, round_inputs

pytestmark = pytest.mark.gpu


def _pair(d, prm, steps, precision, forcing, kernel=tslb.KERNEL_AUTO, jet=None):
    okw = dict(two_component=True, sigma=prm["sigma"], interface_width=prm["W"], forcing=forcing,
               hermite_order=prm.get("order", 3))
    gkw = dict(two_component=True, sigma=prm["sigma"], interface_width=prm["W"], forcing=forcing,
               hermite_order=prm.get("order", 3), kernel=kernel)
    if jet:
        okw.update(bc_zlo=ref.BC_JET_INFLOW, bc_zhi=ref.BC_OUTFLOW, jet_diameter=jet["jet_diameter"],
                   jet_velocity=jet["jet_velocity"], jet_perturbation=jet["jet_perturbation"], seed=jet["seed"])
        gkw.update(jet=True, jet_diameter=jet["jet_diameter"], jet_velocity=jet["jet_velocity"],
                   jet_perturbation=jet["jet_perturbation"], seed=jet["seed"])
    d = round_inputs(d, precision)
    nz, ny, nx = d["rho"].shape
    o = ref.Oracle(nx, ny, nz, prm["omega"], **okw)
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"], d.get("pineq"))
    g = tslb.Tslb(nx, ny, nz, prm["omega"], precision=precision, **gkw)
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"], d.get("pineq"))
    o.step(steps)
    g.step(steps)
    return o, g


def _check(o, g, tol):
    r = o.get_moments()
    m = {k: (None if v is None else np.asarray(v, dtype=np.float64)) for k, v in g.get_moments().items()}
    e = errs(m, r)
    for k, v in e.items():
        assert v <= tol, (k, v, tol, e)
    up_o = o.get_physical_velocity()
    up_g = np.asarray(g.get_physical_velocity(), dtype=np.float64)
    eu = np.abs(up_g - up_o).max() / max(np.abs(up_o).max(), 1e-300)
    assert eu <= tol, ("physical velocity", eu, tol)
    return e, eu, r, up_o


@pytest.mark.parametrize("order", [3, 2])
def test_guo_small_droplets_fp64_100_steps(order):
    d = inputs.droplets_noise(24, seed=5, ndrop=3, rmin=3.0, rmax=5.0, W=3.0, noise=0.01)
    prm = dict(omega=1.7, sigma=0.01, W=3.0, order=order)
    o, g = _pair(d, prm, 100, tslb.F64, tslb.FORCING_GUO)
    assert g.kernel_name == "generic-guo"
    e, eu, r, up = _check(o, g, TOL[tslb.F64])
    print("guo fp64", order, e, eu)
    # the force matters: the stored (bare) and the time-centred velocity differ
    assert np.abs(up[0] - r["ux"]).max() > 1e-6


def test_guo_c3_like_fp32_10_steps():
    """C3 recipe on 64^3 (droplets + velocity noise, omega = 1.95, sigma = 0.005), fp32, 10 steps."""
    d = inputs.droplets_noise(64, seed=12345, ndrop=10, rmin=6.0, rmax=12.0, W=4.0, noise=0.01)
    prm = dict(omega=1.95, sigma=0.005, W=4.0)
    o, g = _pair(d, prm, 10, tslb.F32, tslb.FORCING_GUO)
    e, eu, _, _ = _check(o, g, TOL[tslb.F32])
    print("guo fp32", e, eu)


@pytest.mark.parametrize("precision,steps", [(tslb.F64, 30), (tslb.F32, 10)])
def test_guo_jet_twin(precision, steps):
    """Inflow/outflow planes (F = 0 there, imposed moments) with the developed-jet state."""
    nx, ny, nz = 48, 40, 36
    jet = inputs.jet_params(nx, ny, nz, D=10, U=0.05, Re=500.0, We=20.0, perturbation=0.05, seed=7)
    d = inputs.jet_developed(nx, ny, nz, D=10, ndrop=6)
    prm = dict(omega=jet["omega"], sigma=jet["sigma"], W=4.0)
    o, g = _pair(d, prm, steps, precision, tslb.FORCING_GUO, jet=jet)
    e, eu, _, _ = _check(o, g, TOL[precision])
    print("guo jet", e, eu)


@pytest.mark.parametrize("kernel", [tslb.KERNEL_GENERIC, tslb.KERNEL_TILED])
@pytest.mark.parametrize("precision,steps", [(tslb.F64, 20), (tslb.F32, 10)])
def test_kick_physical_velocity(kernel, precision, steps):
    """KICK: u' - F/(2 rho) with the F of the previous step's phi (read from the other buffer)."""
    d = inputs.droplets_noise(32, 32, 16, seed=9, ndrop=3, rmin=4.0, rmax=6.0, W=4.0, noise=0.01)
    prm = dict(omega=1.6, sigma=0.02, W=4.0)
    o, g = _pair(d, prm, steps, precision, tslb.FORCING_KICK, kernel=kernel)
    e, eu, r, up = _check(o, g, TOL[precision])
    assert np.abs(up[0] - r["ux"]).max() > 1e-6
    # before the first step there is no kick to centre
    g2 = tslb.Tslb(32, 32, 16, 1.6, precision=precision, two_component=True, sigma=0.02, kernel=kernel)
    dd = round_inputs(d, precision)
    g2.init_fields(dd["rho"], dd["ux"], dd["uy"], dd["uz"], dd["phi"])
    assert np.array_equal(g2.get_physical_velocity()[2], g2.get_moments()["uz"])


def test_guo_parameter_errors():
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(32, 32, 32, 1.0, two_component=True, sigma=0.01, forcing=tslb.FORCING_GUO, kernel=tslb.KERNEL_TILED)
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(32, 32, 32, 1.0, forcing=tslb.FORCING_GUO)
    g = tslb.Tslb(32, 32, 32, 1.0, two_component=True, sigma=0.01, forcing=tslb.FORCING_GUO)
    assert g.kernel_name == "generic-guo"
    g.close()

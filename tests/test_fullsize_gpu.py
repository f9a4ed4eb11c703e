"""Parity at BASELINE.json's FULL size (configs[4], 512x512x1536 fp32 jet) in the launch
configuration bench.py times, on sampled outputs the oracle can compute one by one.

After s steps the value at a node depends only on the initial fields within 2s+2 cells of it, so
a (w^3) window cut out of the full-size initial state, stepped by the oracle as a small periodic
box, reproduces the full-size result on the window's interior (margin 2s+2).  The two z boundary
planes are covered by full-x-y slabs stepped by the oracle with the jet boundary conditions.
Error norm: SURVEY N2 over the union of the sampled nodes; fp32 gate 1e-5."""
import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import inputs, tslb

pytestmark = pytest.mark.gpu

STEPS = 2
MARGIN = 2 * STEPS + 2


def _window(t, x0, y0, z0, w):
    import torch
    nz, ny, nx = t.shape
    ix = (torch.arange(x0, x0 + w, device=t.device) % nx)
    iy = (torch.arange(y0, y0 + w, device=t.device) % ny)
    return t[z0:z0 + w][:, iy][:, :, ix].double().cpu().numpy()


# (precision, nz, interior windows, gate).  fp32: BASELINE configs[4] in full.  fp64: the same x-y extent (1024
# tiles, one CTA of up to 255 registers per thread per SM: the launch shape of the fp64 full-size run) and 320
# planes in several z chunks, gate 1e-12.
CASES = {
    "c5-f32": (tslb.F32, 1536, [(242, 242, 60), (498, 500, 700), (250, 3, 114), (20, 250, 370), (262, 236, 498),
                                (236, 262, 1010), (240, 250, 1266)], 1e-5),
    "c5xy-f64": (tslb.F64, 320, [(242, 242, 60), (498, 500, 240), (250, 3, 114), (20, 250, 270), (262, 236, 90),
                                 (240, 250, 246)], 1e-12),
}


@pytest.mark.parametrize("case", sorted(CASES))
def test_c5_full_size_sampled_against_oracle(case):
    import torch
    import bench
    precision, nz, windows, gate = CASES[case]
    tdt = torch.float32 if precision == tslb.F32 else torch.float64
    if torch.cuda.get_device_properties(0).total_memory < 90e9:
        pytest.skip("needs ~75 GB of device memory")
    nx, ny, _, D, _ = bench.CONFIGS["c5"]
    prm = inputs.jet_params(nx, ny, nz, D, We=2000.0)
    dev = torch.device("cuda", 0)
    st = bench.developed_jet_device(torch, nx, ny, nz, D, prm["jet_velocity"], tdt, dev)
    # seeded transverse velocity noise so that every moment is non-trivial
    g = torch.Generator(device=dev).manual_seed(4321)
    for k in ("ux", "uy"):
        st[k] = (torch.rand((nz, ny, nx), generator=g, device=dev, dtype=tdt) - 0.5) * 0.004
    kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
    sim = tslb.Tslb(nx, ny, nz, prm["omega"], precision=precision, **kw)   # same selection as bench.py
    assert "tiled" in sim.kernel_name
    zc = int(sim.kernel_name.split("zc=")[1].rstrip(">"))
    assert zc < nz                     # several z chunks, as in the full-size run
    sim.init_fields(st["rho"], st["ux"], st["uy"], st["uz"], st["phi"])
    sim.step(STEPS)
    out = sim.get_moments(device=True)
    names = ("rho", "ux", "uy", "uz", "phi")
    okw = dict(two_component=True, sigma=prm["sigma"], interface_width=prm["interface_width"])
    num = dict(rho=0.0, u=0.0, pineq=0.0, phi=0.0)
    den = dict(rho=0.0, u=0.0, pineq=0.0, phi=0.0)

    def accumulate(gpu, refm, sl):
        for k in ("rho", "phi"):
            num[k] = max(num[k], np.abs(gpu[k][sl] - refm[k][sl]).max()); den[k] = max(den[k], np.abs(refm[k][sl]).max())
        for k in ("ux", "uy", "uz"):
            num["u"] = max(num["u"], np.abs(gpu[k][sl] - refm[k][sl]).max()); den["u"] = max(den["u"], np.abs(refm[k][sl]).max())
        num["pineq"] = max(num["pineq"], np.abs(gpu["pineq"][(slice(None),) + sl] - refm["pineq"][(slice(None),) + sl]).max())
        den["pineq"] = max(den["pineq"], np.abs(refm["pineq"][(slice(None),) + sl]).max())

    # interior windows: jet core, tile / chunk / periodic edges, core end, downstream cone
    w = 28
    for (x0, y0, z0) in windows:
        ini = {k: _window(st[k], x0, y0, z0, w) for k in names}
        o = ref.Oracle(w, w, w, prm["omega"], **okw)
        o.init_fields(ini["rho"], ini["ux"], ini["uy"], ini["uz"], ini["phi"])
        o.step(STEPS)
        r = o.get_moments()
        o.close()
        gpu = {k: _window(out[k], x0, y0, z0, w) for k in names}
        gpu["pineq"] = np.stack([_window(out["pineq"][c], x0, y0, z0, w) for c in range(6)])
        m = MARGIN
        accumulate(gpu, r, (slice(m, w - m), slice(m, w - m), slice(m, w - m)))

    # boundary slabs (full x-y): inflow at z = 0 and outflow at z = nz-1
    sz = 14
    jet = dict(bc_zlo=ref.BC_JET_INFLOW, bc_zhi=ref.BC_OUTFLOW, jet_diameter=prm["jet_diameter"],
               jet_velocity=prm["jet_velocity"], jet_perturbation=prm["jet_perturbation"], seed=prm["seed"])
    for zlo, keep in ((0, slice(0, sz - MARGIN)), (nz - sz, slice(MARGIN, sz))):
        ini = {k: st[k][zlo:zlo + sz].double().cpu().numpy() for k in names}
        o = ref.Oracle(nx, ny, sz, prm["omega"], **okw, **jet)
        o.init_fields(ini["rho"], ini["ux"], ini["uy"], ini["uz"], ini["phi"])
        if zlo != 0:
            # the slab's own z = 0 plane is not the real inflow plane: it is excluded by `keep`
            pass
        o.step(STEPS)
        r = o.get_moments()
        o.close()
        gpu = {k: out[k][zlo:zlo + sz].double().cpu().numpy() for k in names}
        gpu["pineq"] = np.stack([out["pineq"][c][zlo:zlo + sz].double().cpu().numpy() for c in range(6)])
        accumulate(gpu, r, (keep, slice(None), slice(None)))

    err = {k: num[k] / max(den[k], 1e-300) for k in num}
    print("full-size sampled parity (%s, %d steps):" % (case, STEPS), err, "scales", den)
    assert den["u"] > 0.04 and den["phi"] > 0.99 and den["pineq"] > 1e-6
    for k, v in err.items():
        assert v <= gate, (k, v)
    assert bool(torch.isfinite(out["rho"]).all()) and bool(torch.isfinite(out["phi"]).all())
    sim.close()


@pytest.mark.parametrize("We", [10.0, 200.0, 2000.0])
def test_c4_jet_runs_stay_physical(We):
    """BASELINE configs[3] at full size (256x256x512 fp32, D=20, U=0.05, Re=5000) for the three
    Weber numbers, 2000 steps from rest: properties that hold at any size -- finite fields, phi in
    [0,1] up to a small overshoot, density near 1, the jet tip advancing at about U/2 and the amount
    of injected fluid matching the inlet flux  sum_nozzle U (1 + p xi) per step."""
    import torch
    nx, ny, nz, D, U = 256, 256, 512, 20, 0.05
    prm = inputs.jet_params(nx, ny, nz, D, U=U, Re=5000.0, We=We, perturbation=0.05, seed=2024)
    kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
    sim = tslb.Tslb(nx, ny, nz, prm["omega"], precision=tslb.F32, **kw)
    dev = torch.device("cuda", 0)
    one = torch.ones((nz, ny, nx), dtype=torch.float32, device=dev)
    zero = torch.zeros((nz, ny, nx), dtype=torch.float32, device=dev)
    sim.init_fields(one, zero, zero.clone(), zero.clone(), zero.clone())
    steps = 2000
    sim.step(steps)
    m = sim.get_moments(device=True, want=("rho", "uz", "phi"))
    rho, uz, phi = m["rho"], m["uz"], m["phi"]
    assert bool(torch.isfinite(rho).all()) and bool(torch.isfinite(phi).all()) and bool(torch.isfinite(uz).all())
    assert float(phi.min()) > -0.05 and float(phi.max()) < 1.05
    assert 0.95 < float(rho.min()) and float(rho.max()) < 1.05
    axis = phi[:, ny // 2 - 1:ny // 2 + 1, nx // 2 - 1:nx // 2 + 1].mean(dim=(1, 2)).cpu().numpy()
    tip = int(np.argmax(axis < 0.5))
    assert 0.3 * U * steps < tip < 1.2 * U * steps, tip
    ndisc = sum(1 for x in range(nx) for y in range(ny)
                if (2 * x - (nx - 1)) ** 2 + (2 * y - (ny - 1)) ** 2 < (2 * D / 2) ** 2)
    injected = float(phi[1:].double().sum())
    assert 0.6 * ndisc * U * steps < injected < 1.1 * ndisc * U * steps, (injected, ndisc * U * steps)
    print("We", We, "tip", tip, "injected/expected", injected / (ndisc * U * steps),
          "phi range", float(phi.min()), float(phi.max()), "rho range", float(rho.min()), float(rho.max()))
    sim.close()

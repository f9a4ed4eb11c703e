"""z-slab decomposition (include/tslb.h "z-slabs"): a domain split into slabs whose
step kernels push their face planes into the neighbours' ghost planes must reproduce the
single-context run BIT FOR BIT (same kernels, same arithmetic per node, inflow hash keyed by
(x, y, step)) and therefore agree with the oracle within the usual gates.  One GPU: all slabs
live on device 0 (same stream = the protocol's barrier); the cross-process path (CUDA IPC handles,
host barrier over gloo) runs as two processes sharing the GPU."""
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import ref
from paper_2403_15773_b200 import inputs, slabs, tslb
from tests.test_parity_gpu import TOL, errs, gpu_kwargs, oracle_kwargs, round_inputs

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_single(d, prm, steps, precision, kernel):
    g = tslb.Tslb(prm["nx"], prm["ny"], prm["nz"], prm["omega"], precision=precision, kernel=kernel, **gpu_kwargs(prm))
    g.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
    g.step(steps)
    m = g.get_moments()
    name = g.kernel_name
    g.close()
    return m, name


def run_slabs(d, prm, steps, precision, kernel, n):
    kw = gpu_kwargs(prm)
    s = slabs.LocalSlabs(prm["nx"], prm["ny"], prm["nz"], prm["omega"], n, precision=precision, kernel=kernel, **kw)
    s.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
    s.step(steps)
    m = s.get_moments()
    names = s.kernel_names
    s.close()
    return m, names


def same_bits(a, b):
    for k in ("rho", "ux", "uy", "uz", "pineq", "phi"):
        if a[k] is None:
            assert b[k] is None
            continue
        assert a[k].shape == b[k].shape, k
        assert np.array_equal(a[k], b[k]), (k, np.abs(a[k].astype(np.float64) - b[k]).max())


def oracle(d, prm, steps):
    o = ref.Oracle(prm["nx"], prm["ny"], prm["nz"], prm["omega"], **oracle_kwargs(prm))
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
    o.step(steps)
    r = o.get_moments()
    o.close()
    return r


@pytest.mark.parametrize("kernel", [tslb.KERNEL_TILED, tslb.KERNEL_GENERIC])
@pytest.mark.parametrize("precision", [tslb.F64, tslb.F32])
@pytest.mark.parametrize("n", [1, 2, 3])
def test_periodic_slabs_match_single_context_and_oracle(kernel, precision, n):
    nx, ny, nz = 64, 24, 23                       # 23 planes -> slabs of 8, 8, 7
    prm = dict(nx=nx, ny=ny, nz=nz, omega=1.8, two_component=True, sigma=0.01, interface_width=3.0)
    d = round_inputs(inputs.smooth_random(nx, ny, nz, seed=31), precision)
    steps = 12 if precision == tslb.F64 else 10
    one, name = run_single(d, prm, steps, precision, kernel)
    many, names = run_slabs(d, prm, steps, precision, kernel, n)
    assert all(("tiled" in k) == ("tiled" in name) for k in names)
    same_bits(one, many)
    e = errs({k: (None if v is None else np.asarray(v, dtype=np.float64)) for k, v in many.items()}, oracle(d, prm, steps))
    print("slabs", n, names[0], e)
    for k, v in e.items():
        assert v <= TOL[precision], (k, v)


@pytest.mark.parametrize("kernel", [tslb.KERNEL_TILED, tslb.KERNEL_GENERIC])
@pytest.mark.parametrize("n", [2, 3, 4])
def test_jet_slabs_match_single_context_and_oracle(kernel, n):
    """Inflow plane on the first slab, outflow plane on the last, halo faces in between."""
    nx, ny, nz = 64, 32, 26
    prm = inputs.jet_params(nx, ny, nz, D=9, U=0.04, Re=300.0, We=50.0, perturbation=0.1, seed=5)
    d = round_inputs(inputs.jet_developed(nx, ny, nz, D=9, ndrop=5), tslb.F32)
    one, _ = run_single(d, prm, 10, tslb.F32, kernel)
    many, names = run_slabs(d, prm, 10, tslb.F32, kernel, n)
    same_bits(one, many)
    e = errs({k: np.asarray(v, dtype=np.float64) for k, v in many.items()}, oracle(d, prm, 10))
    print("jet slabs", n, names, e)
    for k, v in e.items():
        assert v <= TOL[tslb.F32], (k, v)


def test_single_component_slabs():
    nx, ny, nz = 32, 16, 12
    prm = dict(nx=nx, ny=ny, nz=nz, omega=1.7)
    d = {k: v for k, v in inputs.smooth_random(nx, ny, nz, seed=3).items() if k != "phi"}
    one, _ = run_single(d, prm, 20, tslb.F64, tslb.KERNEL_TILED)
    many, _ = run_slabs(d, prm, 20, tslb.F64, tslb.KERNEL_TILED, 3)
    same_bits(one, many)


def test_slab_protocol_errors():
    s = tslb.Tslb(32, 8, 6, 1.0, bc_zlo=tslb.BC_HALO, bc_zhi=tslb.BC_HALO)
    z = np.zeros((6, 8, 32), dtype=np.float32)
    s.init_fields(z + 1, z, z, z)
    with pytest.raises(tslb.TslbError):          # no neighbour attached
        s.step(1)
    s.attach_neighbor(0, s)
    s.attach_neighbor(1, s)
    s.halo_push()
    with pytest.raises(tslb.TslbError):          # slabs advance one step per call
        s.step(2)
    s.step(1)
    p = tslb.Tslb(32, 8, 6, 1.0)
    with pytest.raises(tslb.TslbError):          # not a halo face
        p.attach_neighbor(0, s)
    with pytest.raises(tslb.TslbError):          # a halo face cannot pair with a periodic face
        tslb.Tslb(32, 8, 6, 1.0, bc_zlo=tslb.BC_HALO, bc_zhi=tslb.BC_PERIODIC)
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(32, 8, 1, 1.0, bc_zlo=tslb.BC_HALO, bc_zhi=tslb.BC_HALO)
    s.close()
    p.close()


@pytest.mark.parametrize("jet", [False, True])
def test_two_processes_cuda_ipc(tmp_path, jet):
    """One process per slab (RankSlab): CUDA IPC handles exchanged over gloo, host barrier per
    step; the two processes share GPU 0 (their kernels never wait on one another)."""
    out = str(tmp_path / "ipc.npz")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
           "127.0.0.1", "--master-port", "29517", os.path.join(ROOT, "tests", "slab_ipc_worker.py"), out, "1" if jet else "0"]
    env = dict(os.environ, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    z = np.load(out)
    from tests import slab_ipc_worker as w
    d, prm = w.case(jet)
    one, _ = run_single(d, prm, w.STEPS, tslb.F32, tslb.KERNEL_AUTO)
    for k in ("rho", "ux", "uy", "uz", "phi", "pineq"):
        assert np.array_equal(z[k], one[k]), k


# ---------------------------------------------------------------- more than one GPU (skipped on a 1-GPU box)
def _need_two_gpus():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")


@pytest.mark.parametrize("kernel", [tslb.KERNEL_TILED, tslb.KERNEL_GENERIC])
@pytest.mark.parametrize("jet", [False, True])
def test_local_slabs_on_two_devices(kernel, jet):
    """One process, slabs on devices 0 and 1: peer-mapped stores into the neighbour's ghost planes; the
    tiled kernel's dynamic shared-memory attribute has to be set on EACH device."""
    _need_two_gpus()
    from tests import slab_ipc_worker as w
    d, prm = w.case(jet)
    one, _ = run_single(d, prm, w.STEPS, tslb.F32, kernel)
    s = slabs.LocalSlabs(prm["nx"], prm["ny"], prm["nz"], prm["omega"], 2, precision=tslb.F32, devices=[0, 1],
                         kernel=kernel, **gpu_kwargs(prm))
    s.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d.get("phi"), d.get("pineq"))
    s.step(w.STEPS)
    many = s.get_moments()
    s.close()
    same_bits(one, many)


@pytest.mark.parametrize("jet", [False, True])
def test_two_ranks_two_gpus_nccl(tmp_path, jet):
    """One process per GPU (RankSlab): CUDA IPC handles, peer stores across devices, and the per-step
    barrier as a one-element NCCL all-reduce on the library's stream."""
    _need_two_gpus()
    out = str(tmp_path / "nccl.npz")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
           "127.0.0.1", "--master-port", "29519", os.path.join(ROOT, "tests", "slab_ipc_worker.py"), out,
           "1" if jet else "0", "nccl"]
    env = dict(os.environ, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    z = np.load(out)
    from tests import slab_ipc_worker as w
    d, prm = w.case(jet)
    one, _ = run_single(d, prm, w.STEPS, tslb.F32, tslb.KERNEL_AUTO)
    for k in ("rho", "ux", "uy", "uz", "phi", "pineq"):
        assert np.array_equal(z[k], one[k]), k


def test_slab_with_an_imposed_plane_needs_three_planes():
    with pytest.raises(tslb.TslbError, match="nz >= 3"):
        tslb.Tslb(32, 8, 2, 1.0, two_component=True, sigma=0.01, bc_zlo=tslb.BC_JET_INFLOW, bc_zhi=tslb.BC_HALO,
                  jet_diameter=4.0, jet_velocity=0.05, torch_workspace=False)
    with pytest.raises(ValueError):
        slabs.slab_ranges(8, 4, jet=True)
    assert slabs.slab_ranges(12, 4, jet=True) == [(0, 3), (3, 6), (6, 9), (9, 12)]

"""ctypes wrapper of the CPU oracle (oracle/tslb_ref.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg.  Nothing under paper_2403_15773_b200/ imports this and this
imports nothing from there.  Marshalling only -- every step of the method runs in tslb_ref.cpp.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtslb_ref.so")
_SRC = [os.path.join(_HERE, "tslb_ref.cpp"), os.path.join(_HERE, "tslb_ref.h")]

BC_PERIODIC, BC_JET_INFLOW, BC_OUTFLOW = 0, 1, 2
FORCING_KICK, FORCING_GUO = 0, 1


def build(force=False):
    """Compile the oracle with g++ (-O2, no fast-math, OpenMP over z for timing only)."""
    if not force and os.path.exists(_SO) and all(
            os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC[0]]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class _Params(ctypes.Structure):
    _fields_ = [
        ("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
        ("two_component", ctypes.c_int), ("hermite_order", ctypes.c_int),
        ("omega", ctypes.c_double), ("sigma", ctypes.c_double),
        ("interface_width", ctypes.c_double),
        ("bc_zlo", ctypes.c_int), ("bc_zhi", ctypes.c_int),
        ("jet_diameter", ctypes.c_double), ("jet_velocity", ctypes.c_double),
        ("jet_perturbation", ctypes.c_double),
        ("seed", ctypes.c_ulonglong),
        ("forcing", ctypes.c_int),
    ]


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        L.tslb_ref_create.argtypes = [ctypes.POINTER(_Params), ctypes.POINTER(ctypes.c_void_p)]
        L.tslb_ref_init_fields.argtypes = [ctypes.c_void_p, _dp, _dp, _dp, _dp, _dp,
                                           ctypes.POINTER(_dp)]
        L.tslb_ref_step.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.tslb_ref_get_moments.argtypes = [ctypes.c_void_p, _dp, _dp, _dp, _dp,
                                           ctypes.POINTER(_dp), _dp]
        L.tslb_ref_destroy.argtypes = [ctypes.c_void_p]
        L.tslb_ref_lattice.argtypes = [ctypes.POINTER(ctypes.c_int), _dp]
        L.tslb_ref_lattice.restype = None
        L.tslb_ref_feq.argtypes = [ctypes.c_double, _dp, ctypes.c_int, _dp]
        L.tslb_ref_feq.restype = None
        L.tslb_ref_fneq.argtypes = [_dp, _dp, ctypes.c_int, _dp]
        L.tslb_ref_fneq.restype = None
        L.tslb_ref_get_populations.argtypes = [ctypes.c_void_p, _dp]
        L.tslb_ref_phase_geometry.argtypes = [ctypes.c_void_p, _dp, _dp, _dp, _dp]
        L.tslb_ref_set_extra_force.argtypes = [ctypes.c_void_p, _dp]
        L.tslb_ref_get_physical_velocity.argtypes = [ctypes.c_void_p, _dp, _dp, _dp]
        L.tslb_ref_xi.argtypes = [ctypes.c_ulonglong, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                  ctypes.c_int, ctypes.c_longlong]
        L.tslb_ref_xi.restype = ctypes.c_double
        L.tslb_ref_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _c64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def lattice():
    c = np.zeros((27, 3), dtype=np.int32)
    w = np.zeros(27, dtype=np.float64)
    lib().tslb_ref_lattice(c.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), _p(w))
    return c, w


def feq(rho, u, order=3):
    u = _c64(u)
    out = np.zeros(27)
    lib().tslb_ref_feq(float(rho), _p(u), int(order), _p(out))
    return out


def fneq(pineq6, u, order=3):
    pineq6, u = _c64(pineq6), _c64(u)
    out = np.zeros(27)
    lib().tslb_ref_fneq(_p(pineq6), _p(u), int(order), _p(out))
    return out


def xi(seed, x, y, nx, ny, step):
    return lib().tslb_ref_xi(int(seed), int(x), int(y), int(nx), int(ny), int(step))


def num_threads():
    return lib().tslb_ref_num_threads()


class Oracle:
    """One oracle context.  Field arrays have shape (nz, ny, nx) (x fastest), float64."""

    def __init__(self, nx, ny, nz, omega, two_component=False, hermite_order=3, sigma=0.0,
                 interface_width=4.0, bc_zlo=BC_PERIODIC, bc_zhi=BC_PERIODIC, jet_diameter=0.0,
                 jet_velocity=0.0, jet_perturbation=0.0, seed=0, forcing=FORCING_KICK):
        self.shape = (nz, ny, nx)
        self.N = nx * ny * nz
        self.two = bool(two_component)
        self._prm = _Params(nx, ny, nz, int(self.two), hermite_order, omega, sigma,
                            interface_width, bc_zlo, bc_zhi, jet_diameter, jet_velocity,
                            jet_perturbation, seed, int(forcing))
        self._h = ctypes.c_void_p()
        rc = lib().tslb_ref_create(ctypes.byref(self._prm), ctypes.byref(self._h))
        if rc != 0:
            raise ValueError("tslb_ref_create failed: %d" % rc)

    def close(self):
        if self._h:
            lib().tslb_ref_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init_fields(self, rho, ux, uy, uz, phi=None, pineq=None):
        rho, ux, uy, uz, phi = map(_c64, (rho, ux, uy, uz, phi))
        for a in (rho, ux, uy, uz) + ((phi,) if phi is not None else ()):
            assert a.shape == self.shape, (a.shape, self.shape)
        arr = (_dp * 6)()
        keep = []
        if pineq is not None:
            for k in range(6):
                a = _c64(pineq[k])
                assert a.shape == self.shape
                keep.append(a)
                arr[k] = _p(a)
        rc = lib().tslb_ref_init_fields(self._h, _p(rho), _p(ux), _p(uy), _p(uz), _p(phi),
                                        arr if pineq is not None else None)
        if rc != 0:
            raise RuntimeError("tslb_ref_init_fields failed: %d" % rc)

    def step(self, n=1):
        rc = lib().tslb_ref_step(self._h, int(n))
        if rc != 0:
            raise RuntimeError("tslb_ref_step failed: %d" % rc)

    def get_moments(self):
        """-> dict rho, ux, uy, uz, pineq (6, nz, ny, nx), phi (or None)."""
        rho, ux, uy, uz = (np.empty(self.shape) for _ in range(4))
        pin = np.empty((6,) + self.shape)
        phi = np.empty(self.shape) if self.two else None
        arr = (_dp * 6)(*[_p(pin[k]) for k in range(6)])
        rc = lib().tslb_ref_get_moments(self._h, _p(rho), _p(ux), _p(uy), _p(uz), arr, _p(phi))
        if rc != 0:
            raise RuntimeError("tslb_ref_get_moments failed: %d" % rc)
        return dict(rho=rho, ux=ux, uy=uy, uz=uz, pineq=pin, phi=phi)

    def set_extra_force(self, F):
        """Pin-only probe: static force density F (3, nz, ny, nx) added to sigma kappa grad(phi);
        None clears it.  Call before init_fields."""
        if F is None:
            rc = lib().tslb_ref_set_extra_force(self._h, None)
        else:
            F = _c64(F)
            assert F.shape == (3,) + self.shape
            rc = lib().tslb_ref_set_extra_force(self._h, _p(F))
        assert rc == 0

    def get_physical_velocity(self):
        """-> (3, nz, ny, nx): the time-centred velocity (KICK: u' - F/2rho; GUO: u_b + F/2rho)."""
        u = np.empty((3,) + self.shape)
        rc = lib().tslb_ref_get_physical_velocity(self._h, _p(u[0]), _p(u[1]), _p(u[2]))
        assert rc == 0
        return u

    def get_populations(self):
        f = np.empty((27,) + self.shape)
        rc = lib().tslb_ref_get_populations(self._h, _p(f))
        assert rc == 0
        return f

    def phase_geometry(self):
        """-> G (3,...), n (3,...), kappa, F (3,...) of the current phi."""
        G, n, F = (np.empty((3,) + self.shape) for _ in range(3))
        kappa = np.empty(self.shape)
        rc = lib().tslb_ref_phase_geometry(self._h, _p(G), _p(n), _p(kappa), _p(F))
        assert rc == 0
        return G, n, kappa, F

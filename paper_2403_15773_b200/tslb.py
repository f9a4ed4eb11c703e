"""Thin Python binding of the C-ABI CUDA library (include/tslb.h), same names, marshalling only.

PyTorch is used for device memory (workspace, I/O tensors) and streams; every step of the method
runs inside libtslb.so.  There is no CPU fallback: if the library is missing or no B200 is
visible, calls fail loudly.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtslb.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4
F32, F64 = 0, 1
BC_PERIODIC, BC_JET_INFLOW, BC_OUTFLOW, BC_HALO = 0, 1, 2, 3
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED = 0, 1, 2
FORCING_KICK, FORCING_GUO = 0, 1

EXPORTS = ["tslb_workspace_bytes", "tslb_create", "tslb_init_fields", "tslb_step",
           "tslb_get_moments", "tslb_get_physical_velocity", "tslb_get_physical_velocity_noalloc",
           "tslb_noalloc_scratch_bytes", "tslb_step_count", "tslb_kernel_name", "tslb_launch_count",
           "tslb_debug_xi", "tslb_debug_math", "tslb_destroy", "tslb_last_error", "tslb_workspace_ptr",
           "tslb_attach_neighbor", "tslb_ipc_get_handle", "tslb_attach_neighbor_ipc", "tslb_detach_neighbors", "tslb_halo_push",
           "tslb_stats_begin", "tslb_stats_get", "tslb_stats_end"]


class Params(ctypes.Structure):
    """Mirror of `tslb_params` (include/tslb.h)."""
    _fields_ = [
        ("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
        ("precision", ctypes.c_int), ("two_component", ctypes.c_int),
        ("hermite_order", ctypes.c_int),
        ("omega", ctypes.c_double), ("sigma", ctypes.c_double),
        ("interface_width", ctypes.c_double),
        ("bc_zlo", ctypes.c_int), ("bc_zhi", ctypes.c_int),
        ("jet_diameter", ctypes.c_double), ("jet_velocity", ctypes.c_double),
        ("jet_perturbation", ctypes.c_double),
        ("seed", ctypes.c_ulonglong),
        ("device", ctypes.c_int), ("kernel", ctypes.c_int),
        ("stream", ctypes.c_void_p), ("workspace", ctypes.c_void_p),
        ("workspace_bytes", ctypes.c_size_t),
        ("forcing", ctypes.c_int),
    ]


class TslbError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("tslb error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Load libtslb.so (build it with `python -m paper_2403_15773_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError("%s is missing: run `python -m paper_2403_15773_b200.build` "
                              "(there is no CPU fallback)" % _SO)
        L = ctypes.CDLL(_SO)
        vp, pp = ctypes.c_void_p, ctypes.POINTER(Params)
        L.tslb_workspace_bytes.argtypes = [pp]
        L.tslb_workspace_bytes.restype = ctypes.c_size_t
        L.tslb_create.argtypes = [pp, ctypes.POINTER(vp)]
        L.tslb_init_fields.argtypes = [vp, vp, vp, vp, vp, vp, ctypes.POINTER(vp), ctypes.c_int]
        L.tslb_step.argtypes = [vp, ctypes.c_int]
        L.tslb_get_moments.argtypes = [vp, vp, vp, vp, vp, ctypes.POINTER(vp), vp, ctypes.c_int]
        L.tslb_get_physical_velocity.argtypes = [vp, vp, vp, vp, ctypes.c_int]
        L.tslb_get_physical_velocity_noalloc.argtypes = [vp, vp, vp, vp]
        L.tslb_noalloc_scratch_bytes.argtypes = []
        L.tslb_noalloc_scratch_bytes.restype = ctypes.c_size_t
        L.tslb_step_count.argtypes = [vp]
        L.tslb_step_count.restype = ctypes.c_longlong
        L.tslb_kernel_name.argtypes = [vp]
        L.tslb_kernel_name.restype = ctypes.c_char_p
        L.tslb_launch_count.argtypes = [vp]
        L.tslb_launch_count.restype = ctypes.c_longlong
        L.tslb_debug_xi.argtypes = [vp, ctypes.c_longlong, ctypes.POINTER(ctypes.c_double)]
        L.tslb_debug_math.argtypes = [vp, ctypes.c_int] + [ctypes.POINTER(ctypes.c_double)] * 3
        L.tslb_destroy.argtypes = [vp]
        L.tslb_last_error.argtypes = [vp]
        L.tslb_last_error.restype = ctypes.c_char_p
        L.tslb_workspace_ptr.argtypes = [vp]
        L.tslb_workspace_ptr.restype = vp
        L.tslb_attach_neighbor.argtypes = [vp, ctypes.c_int, vp, ctypes.c_int]
        L.tslb_ipc_get_handle.argtypes = [vp, vp]
        L.tslb_attach_neighbor_ipc.argtypes = [vp, ctypes.c_int, vp, ctypes.c_int]
        L.tslb_detach_neighbors.argtypes = [vp]
        L.tslb_halo_push.argtypes = [vp]
        L.tslb_stats_begin.argtypes = [vp, ctypes.c_int]
        L.tslb_stats_get.argtypes = [vp, vp, vp, ctypes.POINTER(ctypes.c_longlong)]
        L.tslb_stats_end.argtypes = [vp]
        _lib = L
    return _lib


def make_params(nx, ny, nz, omega, precision=F32, two_component=False, hermite_order=3, sigma=0.0,
                interface_width=4.0, jet=False, jet_diameter=0.0, jet_velocity=0.0,
                jet_perturbation=0.0, seed=0, device=0, kernel=KERNEL_AUTO, stream=None,
                workspace=None, workspace_bytes=0, bc_zlo=None, bc_zhi=None, forcing=FORCING_KICK):
    """`jet` sets JET_INFLOW/OUTFLOW; bc_zlo / bc_zhi override one face (BC_HALO for a z-slab)."""
    lo = (BC_JET_INFLOW if jet else BC_PERIODIC) if bc_zlo is None else bc_zlo
    hi = (BC_OUTFLOW if jet else BC_PERIODIC) if bc_zhi is None else bc_zhi
    return Params(nx, ny, nz, precision, int(bool(two_component)), hermite_order, omega, sigma,
                  interface_width, lo, hi, jet_diameter, jet_velocity, jet_perturbation,
                  seed, device, kernel, stream, workspace, workspace_bytes, int(forcing))


def workspace_bytes(**kw):
    p = make_params(**kw)
    return lib().tslb_workspace_bytes(ctypes.byref(p))


class Tslb:
    """One simulation context on one GPU.  Field arrays are (nz, ny, nx), x fastest."""

    def __init__(self, nx, ny, nz, omega, precision=F32, torch_workspace=True, **kw):
        import torch
        self._torch = torch
        self.shape = (nz, ny, nx)
        self.precision = precision
        self.two = bool(kw.get("two_component", False))
        self.np_dtype = np.float32 if precision == F32 else np.float64
        self.torch_dtype = torch.float32 if precision == F32 else torch.float64
        dev = kw.get("device", 0)
        self.device = torch.device("cuda", dev)
        p = make_params(nx, ny, nz, omega, precision=precision, **kw)
        if p.stream is None and torch.cuda.is_available():
            with torch.cuda.device(dev):
                p.stream = torch.cuda.current_stream().cuda_stream
        self._ws = None
        if torch_workspace and torch.cuda.is_available():
            nbytes = lib().tslb_workspace_bytes(ctypes.byref(p))
            if nbytes == 0:
                raise TslbError(EINVAL, "invalid parameters")
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            ptr = (self._ws.data_ptr() + 255) // 256 * 256
            p.workspace, p.workspace_bytes = ptr, nbytes
        self.params = p
        self._h = ctypes.c_void_p()
        rc = lib().tslb_create(ctypes.byref(p), ctypes.byref(self._h))
        if rc != OK:
            raise TslbError(rc, lib().tslb_last_error(None).decode())

    # -- helpers
    def _check(self, rc):
        if rc != OK:
            raise TslbError(rc, lib().tslb_last_error(self._h).decode())

    def _ptr(self, a):
        if a is None:
            return None, None
        torch = self._torch
        if isinstance(a, torch.Tensor):
            assert a.dtype == self.torch_dtype and a.is_contiguous() and tuple(a.shape) == self.shape
            return a.data_ptr(), a
        b = np.ascontiguousarray(a, dtype=self.np_dtype)
        assert b.shape == self.shape, (b.shape, self.shape)
        return b.ctypes.data, b

    def close(self):
        if getattr(self, "_h", None):
            lib().tslb_destroy(self._h)
            self._h = ctypes.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the five calls
    def init_fields(self, rho, ux, uy, uz, phi=None, pineq=None):
        """numpy arrays (host pointers) or torch CUDA tensors (device pointers), not mixed."""
        torch = self._torch
        on_dev = isinstance(rho, torch.Tensor) and rho.is_cuda
        keep = []
        ptrs = []
        for a in (rho, ux, uy, uz, phi):
            p, k = self._ptr(a)
            ptrs.append(p)
            keep.append(k)
        arr = None
        if pineq is not None:
            arr = (ctypes.c_void_p * 6)()
            for k in range(6):
                p, kk = self._ptr(pineq[k])
                arr[k] = p
                keep.append(kk)
        self._check(lib().tslb_init_fields(self._h, ptrs[0], ptrs[1], ptrs[2], ptrs[3], ptrs[4],
                                           arr, int(on_dev)))

    def step(self, n=1):
        self._check(lib().tslb_step(self._h, int(n)))

    def get_moments(self, device=False, want=("rho", "ux", "uy", "uz", "pineq", "phi")):
        """-> dict of numpy arrays (or torch CUDA tensors when device=True)."""
        torch = self._torch
        out = {}

        def alloc():
            if device:
                return torch.empty(self.shape, dtype=self.torch_dtype, device=self.device)
            return np.empty(self.shape, dtype=self.np_dtype)

        def ptr(a):
            return a.data_ptr() if device else a.ctypes.data

        ptrs = {}
        for k in ("rho", "ux", "uy", "uz"):
            if k in want:
                out[k] = alloc()
                ptrs[k] = ptr(out[k])
        arr = None
        if "pineq" in want:
            comps = [alloc() for _ in range(6)]
            arr = (ctypes.c_void_p * 6)(*[ptr(a) for a in comps])
        phi = None
        if "phi" in want and self.two:
            phi = alloc()
        self._check(lib().tslb_get_moments(self._h, ptrs.get("rho"), ptrs.get("ux"), ptrs.get("uy"),
                                           ptrs.get("uz"), arr, ptr(phi) if phi is not None else None,
                                           int(device)))
        if "pineq" in want:
            out["pineq"] = torch.stack(comps) if device else np.stack(comps)
        out["phi"] = phi
        return out

    def get_physical_velocity(self, device=False):
        """-> (3, nz, ny, nx) numpy array (or torch CUDA tensor): the time-centred velocity."""
        torch = self._torch
        if device:
            u = torch.empty((3,) + self.shape, dtype=self.torch_dtype, device=self.device)
            ptrs = [u[a].data_ptr() for a in range(3)]
        else:
            u = np.empty((3,) + self.shape, dtype=self.np_dtype)
            ptrs = [u[a].ctypes.data for a in range(3)]
        self._check(lib().tslb_get_physical_velocity(self._h, ptrs[0], ptrs[1], ptrs[2], int(device)))
        return u

    def get_physical_velocity_noalloc(self, out):
        """The same into `out`, a (3, nz, ny, nx) torch CUDA tensor of the context's dtype, through the entry
        point that allocates nothing (built-in scratch array; small grids only).  Asynchronous."""
        assert tuple(out.shape) == (3,) + self.shape and out.dtype == self.torch_dtype and out.is_cuda and out.is_contiguous()
        self._check(lib().tslb_get_physical_velocity_noalloc(self._h, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr()))
        return out

    # -- z-slabs (include/tslb.h "z-slabs")
    @property
    def workspace_ptr(self):
        return lib().tslb_workspace_ptr(self._h)

    def attach_neighbor(self, face, other):
        """Same process: `other` is the Tslb holding the slab behind `face` (0: z low, 1: z high)."""
        self._check(lib().tslb_attach_neighbor(self._h, int(face), other.workspace_ptr, other.shape[0]))

    def ipc_handle(self):
        """64-byte CUDA IPC handle of the workspace (needs torch_workspace=False)."""
        buf = ctypes.create_string_buffer(64)
        self._check(lib().tslb_ipc_get_handle(self._h, buf))
        return buf.raw

    def attach_neighbor_ipc(self, face, handle, nb_nz):
        buf = ctypes.create_string_buffer(bytes(handle), 64)
        self._check(lib().tslb_attach_neighbor_ipc(self._h, int(face), buf, int(nb_nz)))

    def detach_neighbors(self):
        self._check(lib().tslb_detach_neighbors(self._h))

    def halo_push(self):
        self._check(lib().tslb_halo_push(self._h))

    # -- time averages on the mid x-z plane (include/tslb.h)
    def stats_begin(self, every=1):
        self._check(lib().tslb_stats_begin(self._h, int(every)))

    def stats_get(self):
        """-> dict(phi=<phi>(z,x) or None, uz=<u_z>(z,x), nsamples): time averages so far."""
        nz, ny, nx = self.shape
        sp = np.zeros((nz, nx), dtype=np.float64)
        su = np.zeros((nz, nx), dtype=np.float64)
        n = ctypes.c_longlong(0)
        self._check(lib().tslb_stats_get(self._h, sp.ctypes.data if self.two else None, su.ctypes.data, ctypes.byref(n)))
        k = max(1, n.value)
        return dict(phi=sp / k if self.two else None, uz=su / k, nsamples=n.value)

    def stats_end(self):
        self._check(lib().tslb_stats_end(self._h))

    # -- bookkeeping / probes
    @property
    def step_count(self):
        return lib().tslb_step_count(self._h)

    @property
    def kernel_name(self):
        return lib().tslb_kernel_name(self._h).decode()

    @property
    def launch_count(self):
        return lib().tslb_launch_count(self._h)

    def debug_math(self, values):
        """The tiled kernel's reciprocal and square root of `values`, evaluated on the device in the context's
        precision (test probe)."""
        v = np.ascontiguousarray(values, dtype=np.float64).ravel()
        pd = ctypes.POINTER(ctypes.c_double)
        rcp, sq = np.empty_like(v), np.empty_like(v)
        self._check(lib().tslb_debug_math(self._h, int(v.size), v.ctypes.data_as(pd), rcp.ctypes.data_as(pd),
                                          sq.ctypes.data_as(pd)))
        return rcp, sq

    def debug_xi(self, step):
        nz, ny, nx = self.shape
        out = np.empty((ny, nx), dtype=np.float64)
        self._check(lib().tslb_debug_xi(self._h, int(step), out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
        return out

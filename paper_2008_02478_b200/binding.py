"""ctypes binding of libborisdemag.so (include/boris_demag.h).  Argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for
device memory and streams.  There is no CPU fallback: if the shared library is
missing, or there is no CUDA device, the calls raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libborisdemag.so")

_lib = None


class DemagError(RuntimeError):
    pass


def lib():
    """The loaded shared library (raises if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise DemagError(
                f"{LIB_PATH} not found: build it with `python -m paper_2008_02478_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        c_int, c_dbl, c_vp = ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.boris_demag_plan_create.restype = c_vp
        L.boris_demag_plan_create.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl]
        L.boris_demag_plan_create_pbc.restype = c_vp
        L.boris_demag_plan_create_pbc.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl, c_int, c_int, c_int]
        L.boris_demag_tensor_host_pbc.restype = c_int
        L.boris_demag_tensor_host_pbc.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl, c_int, c_int, c_int, c_vp]
        L.boris_demag_plan_destroy.restype = None
        L.boris_demag_plan_destroy.argtypes = [c_vp]
        L.boris_demag_apply.restype = c_int
        L.boris_demag_apply.argtypes = [c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_apply_ex.restype = c_int
        L.boris_demag_apply_ex.argtypes = [c_vp, c_vp, c_vp, ctypes.c_uint, c_vp]
        L.boris_demag_apply_timed.restype = c_int
        L.boris_demag_apply_timed.argtypes = [c_vp, c_vp, c_vp, c_vp, ctypes.POINTER(ctypes.c_float),
                                              ctypes.POINTER(c_int)]
        L.boris_demag_energy.restype = c_int
        L.boris_demag_energy.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_apply_energy.restype = c_int
        L.boris_demag_apply_energy.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_apply_host.restype = c_int
        L.boris_demag_apply_host.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_last_error.restype = ctypes.c_char_p
        L.boris_demag_last_error.argtypes = []
        L.boris_demag_plan_info.restype = c_int
        L.boris_demag_plan_info.argtypes = [c_vp, ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(ctypes.c_longlong),
                                            ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(c_int), ctypes.POINTER(c_int)]
        L.boris_demag_plan_kernel_spectrum.restype = c_int
        L.boris_demag_plan_layout.restype = c_int
        L.boris_demag_plan_layout.argtypes = [c_vp, ctypes.POINTER(c_int), ctypes.POINTER(ctypes.c_longlong),
                                              ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(c_int)]
        L.boris_demag_plan_kernel_spectrum.argtypes = [c_vp, c_vp]
        L.boris_demag_tensor_host.restype = c_int
        L.boris_demag_tensor_host.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl, c_vp]
        L.boris_demag_spectrum_host.restype = c_int
        L.boris_demag_spectrum_host.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl, c_vp]
        L.boris_demag_version.restype = ctypes.c_char_p
        L.boris_demag_version.argtypes = []
        L.boris_llg_create.restype = c_vp
        L.boris_llg_create.argtypes = [c_vp, c_int, c_int, c_int] + [c_dbl] * 7
        L.boris_llg_destroy.restype = None
        L.boris_llg_destroy.argtypes = [c_vp]
        L.boris_llg_set_applied_field.restype = c_int
        L.boris_llg_set_applied_field.argtypes = [c_vp, c_dbl, c_dbl, c_dbl]
        L.boris_llg_effective_field.restype = c_int
        L.boris_llg_effective_field.argtypes = [c_vp, c_vp, c_vp, c_vp]
        L.boris_llg_rk4.restype = c_int
        L.boris_llg_rk4.argtypes = [c_vp, c_vp, c_dbl, c_int, c_vp]
        L.boris_demag_f64_plan_create.restype = c_vp
        L.boris_demag_f64_plan_create.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl, c_int, c_int, c_int]
        L.boris_demag_f64_plan_destroy.restype = None
        L.boris_demag_f64_plan_destroy.argtypes = [c_vp]
        L.boris_demag_f64_apply.restype = c_int
        L.boris_demag_f64_apply.argtypes = [c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_f64_energy.restype = c_int
        L.boris_demag_f64_energy.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_f64_plan_info.restype = c_int
        L.boris_demag_f64_plan_info.argtypes = [c_vp, ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(c_int), ctypes.POINTER(c_int)]
        L.boris_demag_ml_plan_create.restype = c_vp
        L.boris_demag_ml_plan_create.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_vp, c_vp, c_int]
        L.boris_demag_ml_plan_destroy.restype = None
        L.boris_demag_ml_plan_destroy.argtypes = [c_vp]
        L.boris_demag_ml_apply.restype = c_int
        L.boris_demag_ml_apply.argtypes = [c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_ml_energy.restype = c_int
        L.boris_demag_ml_energy.argtypes = [c_vp, c_vp, c_vp, c_vp, c_vp]
        L.boris_demag_ml_pair_tensor_host.restype = c_int
        L.boris_demag_ml_pair_tensor_host.argtypes = [c_int, c_int, c_dbl, c_dbl, c_dbl, c_dbl, c_dbl, c_vp]
        L.boris_demag_plan_mesh.restype = c_int
        L.boris_demag_plan_mesh.argtypes = [c_vp, ctypes.POINTER(c_int), ctypes.POINTER(c_dbl)]
        L.boris_demag_energy_noalloc.restype = c_int
        L.boris_demag_energy_noalloc.argtypes = [c_vp, c_vp, ctypes.c_longlong, c_dbl, c_dbl, c_dbl, c_vp, c_vp]
        L.boris_micro_fp32_rate.restype = c_int
        L.boris_micro_fp32_rate.argtypes = [c_int, ctypes.POINTER(c_dbl)]
        L.boris_micro_segment_bw.restype = c_int
        L.boris_micro_segment_bw.argtypes = [c_int, c_int, ctypes.POINTER(c_dbl)]
        _lib = L
    return _lib


def last_error():
    return lib().boris_demag_last_error().decode()


def _check(rc, what):
    if rc != 0:
        raise DemagError(f"{what} failed ({rc}): {last_error()}")


def version():
    return lib().boris_demag_version().decode()


def tensor_host(nx, ny, nz, hx, hy, hz, images=(0, 0, 0)):
    """boris_demag_tensor_host[_pbc]: the library's real-space tensor, fp64 [6][nz][ny][nx] (host only)."""
    out = np.empty((6, nz, ny, nx), np.float64)
    _check(lib().boris_demag_tensor_host_pbc(nx, ny, nz, hx, hy, hz, *[int(v) for v in images], out.ctypes.data),
           "boris_demag_tensor_host_pbc")
    return out


def spectrum_host(nx, ny, nz, hx, hy, hz):
    """boris_demag_spectrum_host: natural reduced spectrum, fp64 [ncomp][nzr][nyr][nxr] (host only)."""
    ncomp = 6 if nz > 1 else 4
    out = np.empty((ncomp, nz + 1 if nz > 1 else 1, ny + 1, nx + 1), np.float64)
    _check(lib().boris_demag_spectrum_host(nx, ny, nz, hx, hy, hz, out.ctypes.data), "boris_demag_spectrum_host")
    return out


class DemagPlan:
    """boris_demag_plan_create / apply / energy on the current CUDA device.

    M, H are torch CUDA float32 tensors of shape [3, nz, ny, nx] (contiguous).
    """

    def __init__(self, nx, ny, nz, hx, hy, hz, images=(0, 0, 0)):
        """images = (ix, iy, iz): copies of the mesh on each side along x, y, z (boris_demag_plan_create_pbc)."""
        self._h = None
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.h = (float(hx), float(hy), float(hz))
        self.images = tuple(int(v) for v in images)
        if any(self.images):
            h = lib().boris_demag_plan_create_pbc(self.nx, self.ny, self.nz, *self.h, *self.images)
        else:
            h = lib().boris_demag_plan_create(self.nx, self.ny, self.nz, *self.h)
        if not h:
            raise DemagError(f"boris_demag_plan_create failed: {last_error()}")
        self._h = h

    @property
    def shape(self):
        return (3, self.nz, self.ny, self.nx)

    def close(self):
        if self._h:
            lib().boris_demag_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, t, name):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                and tuple(t.shape) == self.shape):
            raise DemagError(f"{name} must be a contiguous CUDA float32 tensor of shape {self.shape}")
        return t.data_ptr()

    @staticmethod
    def _stream(stream):
        import torch
        s = torch.cuda.current_stream() if stream is None else stream
        return s.cuda_stream

    def apply(self, M, H, stream=None):
        """H <- -N * M on `stream` (default: torch's current stream).  Asynchronous."""
        _check(lib().boris_demag_apply(self._h, self._ptr(M, "M"), self._ptr(H, "H"), self._stream(stream)),
               "boris_demag_apply")
        return H

    AOS, ACCUMULATE = 1, 2

    def apply_ex(self, M, H, flags, stream=None):
        """boris_demag_apply_ex: AOS -> M, H are [nz][ny][nx][3]; ACCUMULATE -> H += -N * M.  Asynchronous."""
        import torch
        shape = (self.nz, self.ny, self.nx, 3) if flags & self.AOS else self.shape
        for t, name in ((M, "M"), (H, "H")):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                    and tuple(t.shape) == tuple(shape)):
                raise DemagError(f"{name} must be a contiguous CUDA float32 tensor of shape {shape}")
        _check(lib().boris_demag_apply_ex(self._h, M.data_ptr(), H.data_ptr(), int(flags), self._stream(stream)),
               "boris_demag_apply_ex")
        return H

    # timing slots of boris_demag_apply_timed, named per kernel path (boris_demag_plan_layout)
    KINDS = {0: ("XFwd", "Y2D", "YFwd", "ZFused", "YInv", "XInv"),
             2: ("XFwdT", "YFused", "-", "-", "-", "XInvT"),
             3: ("XZFwd", "YFused", "-", "-", "-", "ZXInv"),
             4: ("XFwdT", "YZFused", "-", "-", "-", "XInvP")}

    def apply_timed(self, M, H, stream=None):
        """boris_demag_apply_timed: {kind: (ms, launches)} of one evaluation.  Synchronous."""
        ms = (ctypes.c_float * 6)()
        nl = (ctypes.c_int * 6)()
        _check(lib().boris_demag_apply_timed(self._h, self._ptr(M, "M"), self._ptr(H, "H"), self._stream(stream),
                                             ms, nl), "boris_demag_apply_timed")
        return {k: (ms[i], nl[i]) for i, k in enumerate(self.KINDS[self.layout()["path"]]) if nl[i]}

    def layout(self):
        """boris_demag_plan_layout: kernel path, intermediate spectrum bytes, stored kernel bytes, tile columns."""
        path, cols = ctypes.c_int(), ctypes.c_int()
        sb, kb = ctypes.c_longlong(), ctypes.c_longlong()
        _check(lib().boris_demag_plan_layout(self._h, ctypes.byref(path), ctypes.byref(sb), ctypes.byref(kb),
                                             ctypes.byref(cols)), "boris_demag_plan_layout")
        return {"path": path.value, "spectrum_bytes": sb.value, "kernel_storage_bytes": kb.value, "cols": cols.value}

    def energy(self, M, H, E=None, stream=None):
        """E (CUDA float64 tensor of 1 element) <- -(mu0/2) dV sum M.H.  Asynchronous."""
        import torch
        if E is None:
            E = torch.empty(1, dtype=torch.float64, device=M.device)
        _check(lib().boris_demag_energy(self._h, self._ptr(M, "M"), self._ptr(H, "H"), E.data_ptr(),
                                        self._stream(stream)), "boris_demag_energy")
        return E

    def apply_energy(self, M, H, E=None, stream=None):
        """boris_demag_apply_energy: H <- -N * M and E <- -(mu0/2) dV sum M.H in one enqueue.  Asynchronous."""
        import torch
        if E is None:
            E = torch.empty(1, dtype=torch.float64, device=M.device)
        _check(lib().boris_demag_apply_energy(self._h, self._ptr(M, "M"), self._ptr(H, "H"), E.data_ptr(),
                                              self._stream(stream)), "boris_demag_apply_energy")
        return E

    def apply_host(self, M_host, H_host, want_energy=True, stream=None):
        """Host-buffer entry point: numpy/torch CPU float32 arrays [3][nz][ny][nx]; returns E (float) or None."""
        mp, hp = _host_ptr(M_host, self.shape), _host_ptr(H_host, self.shape)
        e = ctypes.c_double(0.0)
        _check(lib().boris_demag_apply_host(self._h, mp, hp, ctypes.addressof(e) if want_energy else None,
                                            self._stream(stream)), "boris_demag_apply_host")
        return e.value if want_energy else None

    def info(self):
        comp, des, ws = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong()
        padded = (ctypes.c_int * 3)()
        nl = ctypes.c_int()
        _check(lib().boris_demag_plan_info(self._h, ctypes.byref(comp), ctypes.byref(des), ctypes.byref(ws), padded,
                                           ctypes.byref(nl)), "boris_demag_plan_info")
        lay = self.layout()
        return {"compulsory_bytes": comp.value, "designed_hbm_bytes": des.value, "workspace_bytes": ws.value,
                "padded": tuple(padded), "kernel_launches": nl.value, **lay}

    def mesh(self):
        """((nx, ny, nz), (hx, hy, hz)) the plan was created for."""
        cells, sides = (ctypes.c_int * 3)(), (ctypes.c_double * 3)()
        _check(lib().boris_demag_plan_mesh(self._h, cells, sides), "boris_demag_plan_mesh")
        return tuple(cells), tuple(sides)

    def kernel_spectrum(self):
        """Natural reduced fp32 spectrum [ncomp][nzr][nyr][nxr] read back from the device."""
        ncomp = 6 if self.nz > 1 else 4
        Px, Py, Pz = self.info()["padded"]          # of the power-of-two mesh the kernels work on
        out = np.empty((ncomp, Pz // 2 + 1 if self.nz > 1 else 1, Py // 2 + 1, Px // 2 + 1), np.float32)
        _check(lib().boris_demag_plan_kernel_spectrum(self._h, out.ctypes.data), "boris_demag_plan_kernel_spectrum")
        return out


def _host_ptr(a, shape):
    try:
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous() or tuple(a.shape) != tuple(shape):
                raise DemagError(f"host tensor must be contiguous CPU float32 of shape {shape}")
            return a.data_ptr()
    except ImportError:
        pass
    if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous and a.shape == tuple(shape)):
        raise DemagError(f"host array must be C-contiguous float32 of shape {shape}")
    return a.ctypes.data


class LLG:
    """include/boris_llg.h: effective field (demag + exchange + applied field) and RK4 steps of the LLG equation
    on CUDA float32 unit fields [3][nz][ny][nx].  Argument marshalling only."""

    GAMMA = 2.212761569e5          # mu0 |gamma_e|, m / (A s)

    def __init__(self, plan, Ms, A, alpha, gamma=GAMMA, Hext=(0.0, 0.0, 0.0)):
        self.plan = plan
        self._h = lib().boris_llg_create(plan._h, plan.nx, plan.ny, plan.nz, *plan.h, Ms, A, alpha, gamma)
        if not self._h:
            raise DemagError("boris_llg_create failed: " + last_error())
        self.set_applied_field(*Hext)

    def set_applied_field(self, Hx, Hy, Hz):
        _check(lib().boris_llg_set_applied_field(self._h, Hx, Hy, Hz), "boris_llg_set_applied_field")

    def effective_field(self, m, Heff, stream=None):
        _check(lib().boris_llg_effective_field(self._h, self.plan._ptr(m, "m"), self.plan._ptr(Heff, "Heff"),
                                               self.plan._stream(stream)), "boris_llg_effective_field")
        return Heff

    def rk4(self, m, dt, nsteps=1, stream=None):
        _check(lib().boris_llg_rk4(self._h, self.plan._ptr(m, "m"), dt, nsteps, self.plan._stream(stream)), "boris_llg_rk4")
        return m

    def close(self):
        if self._h:
            lib().boris_llg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ----------------------------------------------------------------- fp64 variant (include/boris_demag_f64.h)
class DemagPlanF64:
    """boris_demag_f64_plan_create / apply / energy.  M, H: torch CUDA float64 tensors [3, nz, ny, nx] (contiguous)."""

    def __init__(self, nx, ny, nz, hx, hy, hz, images=(0, 0, 0)):
        self._h = None
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.h = (float(hx), float(hy), float(hz))
        h = lib().boris_demag_f64_plan_create(self.nx, self.ny, self.nz, *self.h, *[int(v) for v in images])
        if not h:
            raise DemagError(f"boris_demag_f64_plan_create failed: {last_error()}")
        self._h = h

    def close(self):
        if self._h:
            lib().boris_demag_f64_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, t, name):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and tuple(t.shape) == (3, self.nz, self.ny, self.nx)):
            raise DemagError(f"{name} must be a contiguous CUDA float64 tensor of shape {(3, self.nz, self.ny, self.nx)}")
        return t.data_ptr()

    @staticmethod
    def _stream(stream):
        import torch
        return (stream or torch.cuda.current_stream()).cuda_stream

    def apply(self, M, H, stream=None):
        _check(lib().boris_demag_f64_apply(self._h, self._ptr(M, "M"), self._ptr(H, "H"), self._stream(stream)),
               "boris_demag_f64_apply")
        return H

    def energy(self, M, H, stream=None):
        import torch
        E = torch.zeros(1, dtype=torch.float64, device=M.device)
        _check(lib().boris_demag_f64_energy(self._h, self._ptr(M, "M"), self._ptr(H, "H"), E.data_ptr(),
                                            self._stream(stream)), "boris_demag_f64_energy")
        return E

    def info(self):
        ws, nl = ctypes.c_longlong(), ctypes.c_int()
        padded = (ctypes.c_int * 3)()
        _check(lib().boris_demag_f64_plan_info(self._h, ctypes.byref(ws), padded, ctypes.byref(nl)), "boris_demag_f64_plan_info")
        return {"workspace_bytes": ws.value, "padded": tuple(padded), "kernel_launches": nl.value}


# ----------------------------------------------------------------- multi-layered convolution (include/boris_demag_ml.h)
def ml_pair_tensor_host(nx, ny, hx, hy, tk, ti, Z):
    """boris_demag_ml_pair_tensor_host: the library's tensor between unequal cuboids, fp64 [6][ny][nx] (host only)."""
    out = np.empty((6, ny, nx), np.float64)
    _check(lib().boris_demag_ml_pair_tensor_host(nx, ny, hx, hy, tk, ti, Z, out.ctypes.data), "boris_demag_ml_pair_tensor_host")
    return out


class MultiLayerPlan:
    """boris_demag_ml_plan_create / apply / energy.  M, H: torch CUDA tensors [3, nlayers, ny, nx], float32 or (fp64=True)
    float64, contiguous.  thickness, z_centre: per-layer cell height and centre height in metres."""

    def __init__(self, nx, ny, hx, hy, thickness, z_centre, fp64=False):
        self._h = None
        t = np.ascontiguousarray(thickness, np.float64)
        z = np.ascontiguousarray(z_centre, np.float64)
        if t.ndim != 1 or t.shape != z.shape:
            raise DemagError("thickness and z_centre must be 1-D arrays of the same length")
        self.nx, self.ny, self.n, self.fp64 = int(nx), int(ny), int(t.size), bool(fp64)
        h = lib().boris_demag_ml_plan_create(self.nx, self.ny, self.n, float(hx), float(hy), t.ctypes.data, z.ctypes.data,
                                             1 if fp64 else 0)
        if not h:
            raise DemagError(f"boris_demag_ml_plan_create failed: {last_error()}")
        self._h = h

    def close(self):
        if self._h:
            lib().boris_demag_ml_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, t, name):
        import torch
        want = torch.float64 if self.fp64 else torch.float32
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == want and t.is_contiguous()
                and tuple(t.shape) == (3, self.n, self.ny, self.nx)):
            raise DemagError(f"{name} must be a contiguous CUDA {want} tensor of shape {(3, self.n, self.ny, self.nx)}")
        return t.data_ptr()

    def apply(self, M, H, stream=None):
        import torch
        st = (stream or torch.cuda.current_stream()).cuda_stream
        _check(lib().boris_demag_ml_apply(self._h, self._ptr(M, "M"), self._ptr(H, "H"), st), "boris_demag_ml_apply")
        return H

    def energy(self, M, H, stream=None):
        import torch
        st = (stream or torch.cuda.current_stream()).cuda_stream
        E = torch.zeros(1, dtype=torch.float64, device=M.device)
        _check(lib().boris_demag_ml_energy(self._h, self._ptr(M, "M"), self._ptr(H, "H"), E.data_ptr(), st),
               "boris_demag_ml_energy")
        return E


# ----------------------------------------------------------------- no allocation (include/boris_demag_noalloc.h)
NOALLOC_MAX_VALUES = 1 << 27


def energy_noalloc(M, H, h, E, stream=None):
    """boris_demag_energy_noalloc: E[0] <- -(mu0/2) hx hy hz sum M.H with the reduction scratch in the library's static
    device array (no plan, no allocation: E is the caller's CUDA float64 tensor).  Asynchronous; calls that overlap on
    the GPU race on the shared array."""
    import torch
    for t, name in ((M, "M"), (H, "H")):
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
            raise DemagError(f"{name} must be a contiguous CUDA float32 tensor")
    if M.numel() != H.numel():
        raise DemagError("M and H must have the same number of elements")
    if not (E.is_cuda and E.dtype == torch.float64 and E.numel() >= 1):
        raise DemagError("E must be a CUDA float64 tensor")
    st = (stream or torch.cuda.current_stream()).cuda_stream
    _check(lib().boris_demag_energy_noalloc(M.data_ptr(), H.data_ptr(), M.numel(), float(h[0]), float(h[1]), float(h[2]),
                                            E.data_ptr(), st), "boris_demag_energy_noalloc")
    return E


# ----------------------------------------------------------------- device probes (include/boris_micro.h)
def micro_fp32_rate(op):
    """Lane operations per second of FADD (0), FFMA (1), FADD2 (2) or FFMA2 (3) over the whole device."""
    out = ctypes.c_double(0.0)
    rc = lib().boris_micro_fp32_rate(int(op), ctypes.byref(out))
    if rc:
        raise DemagError(f"boris_micro_fp32_rate failed ({rc}): {last_error()}")
    return out.value


def micro_segment_bw(seg_bytes, write):
    """GB/s of a read (write = False) or write stream that touches HBM in pieces of seg_bytes."""
    out = ctypes.c_double(0.0)
    rc = lib().boris_micro_segment_bw(int(seg_bytes), 1 if write else 0, ctypes.byref(out))
    if rc:
        raise DemagError(f"boris_micro_segment_bw failed ({rc}): {last_error()}")
    return out.value

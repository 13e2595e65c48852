"""ctypes binding of libugks (include/ugks.h).  Same names as the C ABI, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libugks.so")
_lib = None
_dp = C.POINTER(C.c_double)

EXPORTS = ["ugks_workspace_bytes", "ugks_init", "ugks_set_state", "ugks_step", "ugks_moments", "ugks_get_f",
           "ugks_residual", "ugks_sync", "ugks_dt", "ugks_mu_ref", "ugks_step_count", "ugks_launch_count",
           "ugks_set_option", "ugks_kernel_times", "ugks_jit_check", "ugks_last_error", "ugks_version", "ugks_destroy",
           "ugks_residual_noalloc"]
NOALLOC_MAX_CELLS = 1048576            # UGKS_NOALLOC_MAX_CELLS of include/ugks.h


class UgksError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libugks error {code}: {msg}")
        self.code = code


class _Mesh(C.Structure):
    _fields_ = [("I", C.c_int), ("J", C.c_int), ("x0", C.c_double), ("x1", C.c_double),
                ("y0", C.c_double), ("y1", C.c_double)]


class _VGrid(C.Structure):
    _fields_ = [("Nu", C.c_int), ("Nv", C.c_int), ("u", _dp), ("wu", _dp), ("v", _dp), ("wv", _dp)]


class _Gas(C.Structure):
    _fields_ = [("omega", C.c_double), ("mu_ref", C.c_double), ("Kn", C.c_double), ("Pr", C.c_double),
                ("K_int", C.c_int)]


class _BC(C.Structure):
    _fields_ = [("type", C.c_int), ("rho", C.c_double), ("U", C.c_double), ("V", C.c_double), ("T", C.c_double)]


class _BCs(C.Structure):
    _fields_ = [("xmin", _BC), ("xmax", _BC), ("ymin", _BC), ("ymax", _BC)]


def library_path() -> str:
    return _SO


def lib():
    """Load libugks.so (built in-tree by ``python -m paper_1810_08137_b200.build``).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} not built: run `python -m paper_1810_08137_b200.build` (there is no fallback path)")
        L = C.CDLL(_SO)
        vp = C.c_void_p
        L.ugks_workspace_bytes.argtypes = [C.POINTER(_Mesh), C.POINTER(_VGrid)]; L.ugks_workspace_bytes.restype = C.c_size_t
        L.ugks_init.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.POINTER(_VGrid), C.POINTER(_Gas), C.POINTER(_BCs),
                                C.c_double, vp, C.c_size_t, vp]
        L.ugks_set_state.argtypes = [vp, vp, vp, C.c_int]
        L.ugks_step.argtypes = [vp, C.c_int]
        L.ugks_moments.argtypes = [vp, vp, vp, C.c_int]
        L.ugks_get_f.argtypes = [vp, vp, C.c_int]
        L.ugks_residual.argtypes = [vp, _dp]
        L.ugks_sync.argtypes = [vp]
        L.ugks_dt.argtypes = [vp]; L.ugks_dt.restype = C.c_double
        L.ugks_mu_ref.argtypes = [vp]; L.ugks_mu_ref.restype = C.c_double
        L.ugks_step_count.argtypes = [vp]; L.ugks_step_count.restype = C.c_long
        L.ugks_launch_count.argtypes = [vp]; L.ugks_launch_count.restype = C.c_long
        L.ugks_set_option.argtypes = [vp, C.c_char_p, C.c_int]
        L.ugks_kernel_times.argtypes = [vp, _dp, C.POINTER(C.c_long)]
        L.ugks_jit_check.argtypes = [C.POINTER(_Mesh), C.POINTER(_VGrid), C.POINTER(_BCs), C.c_char_p, C.c_size_t]
        L.ugks_last_error.argtypes = [vp]; L.ugks_last_error.restype = C.c_char_p
        L.ugks_version.argtypes = []; L.ugks_version.restype = C.c_char_p
        L.ugks_destroy.argtypes = [vp]; L.ugks_destroy.restype = None
        L.ugks_residual_noalloc.argtypes = [vp, vp, C.c_long, vp, vp, C.c_char_p, C.c_size_t]
        _lib = L
    return _lib


def _structs(p):
    keep = [np.ascontiguousarray(np.asarray(a, dtype=np.float64)) for a in (p.u, p.wu, p.v, p.wv)]
    mesh = _Mesh(p.I, p.J, p.x0, p.x1, p.y0, p.y1)
    vg = _VGrid(len(keep[0]), len(keep[2]), *[a.ctypes.data_as(_dp) for a in keep])
    gas = _Gas(p.omega, p.mu_ref, p.Kn, p.Pr, p.K_int)
    bcs = _BCs(*[_BC(int(b[0]), float(b[1]), float(b[2]), float(b[3]), float(b[4])) for b in p.bcs])
    return keep, mesh, vg, gas, bcs


def jit_check(problem) -> str:
    """Compile the run-time specialised kernels for ``problem``'s geometry without a device (ugks_jit_check); returns the
    compiler log (ptxas register / shared-memory lines).  Raises on a compile error."""
    keep, mesh, vg, gas, bcs = _structs(problem)
    buf = C.create_string_buffer(1 << 16)
    rc = lib().ugks_jit_check(C.byref(mesh), C.byref(vg), C.byref(bcs), buf, len(buf))
    if rc:
        raise UgksError(rc, buf.value.decode(errors="replace")[-2000:])
    return buf.value.decode(errors="replace")


def workspace_bytes(problem) -> int:
    keep, mesh, vg, gas, bcs = _structs(problem)
    return int(lib().ugks_workspace_bytes(C.byref(mesh), C.byref(vg)))


def residual_noalloc(W_old, W_new, out=None, stream=None):
    """ugks_residual_noalloc: the O11 residual between two W fields [..][4] (float64 torch CUDA tensors) without a context,
    a workspace or any device allocation inside the library -- for code that cannot allocate (a monitoring hook in a
    process whose device memory belongs to a pool, a loop that cannot take cudaMalloc's device-wide synchronisation).
    The partial sums go to a fixed 512 KiB array inside libugks.so that all calls on a device share: keep calls ordered on
    one stream.  ``out``: CUDA tensor of 4 doubles written asynchronously on ``stream`` (default: torch's current stream);
    if None one is made HERE by torch (outside the library) and returned.  At most NOALLOC_MAX_CELLS cells."""
    import torch
    assert W_old.is_cuda and W_new.is_cuda and W_old.dtype == W_new.dtype == torch.float64
    assert W_old.is_contiguous() and W_new.is_contiguous() and W_old.shape == W_new.shape and W_old.shape[-1] == 4
    if out is None:
        out = torch.empty(4, dtype=torch.float64, device=W_new.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 4
    st = stream if stream is not None else torch.cuda.current_stream(W_new.device)
    buf = C.create_string_buffer(320)
    with torch.cuda.device(W_new.device):
        rc = lib().ugks_residual_noalloc(C.c_void_p(W_old.data_ptr()), C.c_void_p(W_new.data_ptr()), W_new.numel() // 4,
                                         C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream), buf, len(buf))
    if rc:
        raise UgksError(rc, buf.value.decode(errors="replace"))
    return out


class Ugks:
    """One libugks context on the current CUDA device and stream.  ``problem``: plain data with the fields of
    ``ugks_mesh / ugks_vgrid / ugks_gas / ugks_bcs`` (see workloads.Problem).  Arrays passed to set_state / returned
    by f(), W() are torch CUDA tensors or numpy arrays; only their pointers cross the ABI."""

    def __init__(self, problem, device="cuda:0", stream=None, tangential=False):
        import torch
        if not torch.cuda.is_available():
            raise UgksError(3, "no CUDA device: libugks has no CPU fallback")
        L = lib()
        self._torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.I, self.J, self.Nu, self.Nv = problem.I, problem.J, len(problem.u), len(problem.v)
        self.N = self.Nu * self.Nv
        keep, mesh, vg, gas, bcs = _structs(problem)
        nbytes = int(L.ugks_workspace_bytes(C.byref(mesh), C.byref(vg)))
        if nbytes == 0:
            raise UgksError(1, "invalid mesh / velocity grid")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = L.ugks_init(C.byref(h), C.byref(mesh), C.byref(vg), C.byref(gas), C.byref(bcs), float(problem.cfl),
                         C.c_void_p(self.workspace.data_ptr()), nbytes, C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise UgksError(rc, L.ugks_last_error(None).decode())
        self._h = h
        if tangential:
            self.set_option("tangential", 1)

    def _chk(self, rc):
        if rc:
            raise UgksError(rc, lib().ugks_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().ugks_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, a, n):
        """(pointer, on_device) of a float64 torch tensor or numpy array holding n doubles, contiguous."""
        torch = self._torch
        if isinstance(a, torch.Tensor):
            assert a.dtype == torch.float64 and a.is_contiguous() and a.numel() == n, (a.dtype, a.shape, n)
            return C.c_void_p(a.data_ptr()), int(a.is_cuda)
        assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n
        return C.c_void_p(a.ctypes.data), 0

    @property
    def dt(self): return lib().ugks_dt(self._h)

    @property
    def mu_ref(self): return lib().ugks_mu_ref(self._h)

    @property
    def step_count(self): return lib().ugks_step_count(self._h)

    @property
    def launch_count(self): return lib().ugks_launch_count(self._h)

    def set_option(self, name, value):
        self._chk(lib().ugks_set_option(self._h, name.encode(), int(value)))

    KERNELS = ("cell_moments", "face_scalars", "cell_scalars", "tables", "flux_update")

    def kernel_times(self):
        """{kernel: (total ms, launches)} since the last call (needs set_option("profile", 1))."""
        ms = np.zeros(5)
        cnt = (C.c_long * 5)()
        self._chk(lib().ugks_kernel_times(self._h, ms.ctypes.data_as(_dp), cnt))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(self.KERNELS)}

    def set_state(self, W, f):
        pw, dw = self._ptr(W, self.I * self.J * 4)
        pf, df = self._ptr(f, self.I * self.J * self.N)
        assert dw == df, "W and f must both be host or both be device arrays"
        self._chk(lib().ugks_set_state(self._h, pw, pf, dw))

    def step(self, n=1):
        self._chk(lib().ugks_step(self._h, int(n)))

    def sync(self):
        self._chk(lib().ugks_sync(self._h))

    def residual(self):
        o = np.empty(4)
        self._chk(lib().ugks_residual(self._h, o.ctypes.data_as(_dp)))
        return o

    def W(self, out=None):
        if out is None:
            out = np.empty((self.J, self.I, 4))
        p, d = self._ptr(out, self.I * self.J * 4)
        self._chk(lib().ugks_moments(self._h, p, None, d))
        return out

    def W_of_f(self, out=None):
        if out is None:
            out = np.empty((self.J, self.I, 4))
        p, d = self._ptr(out, self.I * self.J * 4)
        self._chk(lib().ugks_moments(self._h, None, p, d))
        return out

    def f(self, out=None):
        if out is None:
            out = np.empty((self.J, self.I, self.Nv, self.Nu))
        p, d = self._ptr(out, self.I * self.J * self.N)
        self._chk(lib().ugks_get_f(self._h, p, d))
        return out

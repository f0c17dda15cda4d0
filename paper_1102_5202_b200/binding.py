"""ctypes binding of libhz.so.  Same names as include/hz.h; argument marshalling only."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
HZ_F32, HZ_F64, HZ_F32_F64 = 0, 1, 2
HZ_BC_PERIODIC, HZ_BC_OUTFLOW, HZ_BC_EXTERNAL, HZ_BC_EXTERNAL_OUTFLOW, HZ_BC_OUTFLOW_EXTERNAL = 0, 1, 2, 3, 4
HZ_HALO_PRIM, HZ_HALO_METRIC = 0, 1
HZ_OK, HZ_EINVAL, HZ_ENOMEM, HZ_ECUDA, HZ_ESTATE, HZ_ELIMIT = 0, -1, -2, -3, -4, -5
HZ_NOALLOC_MAX_BLOCKS, HZ_NOALLOC_MAX_FIELDS, HZ_NOALLOC_MAX_CELLS = 1184, 16, 1 << 31

# every symbol include/hz.h declares (tests check the library exports each of them)
SYMBOLS = ["hz_default_params", "hz_state_bytes", "hz_state_bytes_for", "hz_create", "hz_destroy", "hz_set_stream", "hz_set_metric",
           "hz_set_primitives", "hz_step", "hz_substeps", "hz_get_primitives", "hz_get_psi", "hz_get_conserved",
           "hz_diagnostics", "hz_noalloc_setup", "hz_sum_fields_noalloc", "hz_halo_bytes", "hz_halo_pack", "hz_halo_unpack", "hz_prim_buffers", "hz_peer_attach", "hz_peer_detach", "hz_launch_count", "hz_fma_peak", "hz_profile", "hz_profile_read", "hz_kernel_name",
           "hz_strerror"]
HZ_NKERNELS = 2


class HzGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double), ("bc", C.c_int * 3)]


class HzParams(C.Structure):
    _fields_ = [("gamma_ad", C.c_double), ("rho_atm", C.c_double), ("p_atm", C.c_double), ("atm_tol", C.c_double),
                ("cleaning", C.c_int), ("kappa", C.c_double), ("c2p_maxit", C.c_int), ("c2p_tol", C.c_double),
                ("c2p_scheme", C.c_int), ("energy_var", C.c_int), ("recon", C.c_int)]

    @classmethod
    def default(cls, **kw):
        p = cls()
        lib().hz_default_params(C.byref(p))
        for k, v in kw.items():
            if not hasattr(p, k):
                raise AttributeError(k)
            setattr(p, k, v)
        return p


class HzDiag(C.Structure):
    _fields_ = [("sumD", C.c_double), ("sumSx", C.c_double), ("sumSy", C.c_double), ("sumSz", C.c_double),
                ("sumTau", C.c_double), ("sumBx", C.c_double), ("sumBy", C.c_double), ("sumBz", C.c_double),
                ("sumPsi", C.c_double), ("divB_max", C.c_double), ("divB_L1", C.c_double),
                ("max_speed_over_dx", C.c_double), ("c2p_fail", C.c_longlong), ("atm_reset", C.c_longlong),
                ("p_floor", C.c_longlong), ("c2p_maxit_seen", C.c_int), ("c2p_stalled", C.c_longlong)]

    def asdict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class HzError(RuntimeError):
    def __init__(self, code, where=""):
        self.code = code
        try:
            msg = lib().hz_strerror(code).decode()
        except Exception:
            msg = "?"
        super().__init__(f"{where}: hz error {code}: {msg}")


_lib = None


def lib_path():
    return os.path.join(HERE, "libhz.so")


def lib():
    """Load libhz.so (built in-tree by paper_1102_5202_b200/build.py).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: run `python -m paper_1102_5202_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(path)
        vp, ip = C.c_void_p, C.c_int
        L.hz_default_params.argtypes = [C.POINTER(HzParams)]
        L.hz_state_bytes.argtypes = [C.POINTER(HzGrid), ip, C.POINTER(C.c_size_t)]
        L.hz_state_bytes_for.argtypes = [C.POINTER(HzGrid), ip, C.POINTER(HzParams), C.POINTER(C.c_size_t)]
        L.hz_create.argtypes = [C.POINTER(HzGrid), ip, C.POINTER(HzParams), vp, C.POINTER(vp)]
        L.hz_destroy.argtypes = [vp]
        L.hz_set_stream.argtypes = [vp, vp]
        L.hz_set_metric.argtypes = [vp, vp, vp, vp]
        L.hz_set_primitives.argtypes = [vp, vp]
        L.hz_step.argtypes = [vp, C.c_double, ip]
        L.hz_substeps.argtypes = [vp, C.c_double, ip]
        L.hz_get_primitives.argtypes = [vp, vp]
        L.hz_get_psi.argtypes = [vp, vp]
        L.hz_get_conserved.argtypes = [vp, vp]
        L.hz_diagnostics.argtypes = [vp, C.POINTER(HzDiag)]
        L.hz_halo_bytes.argtypes = [vp, ip, C.POINTER(C.c_size_t)]
        L.hz_halo_pack.argtypes = [vp, ip, ip, vp]
        L.hz_halo_unpack.argtypes = [vp, ip, ip, vp]
        L.hz_prim_buffers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_longlong)]
        L.hz_peer_attach.argtypes = [vp, ip, vp, vp, C.c_longlong, ip]
        L.hz_peer_detach.argtypes = [vp, ip]
        L.hz_fma_peak.argtypes = [ip, C.POINTER(C.c_double)]
        L.hz_launch_count.argtypes = [vp]
        L.hz_launch_count.restype = C.c_longlong
        L.hz_profile.argtypes = [vp, ip]
        L.hz_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.hz_kernel_name.argtypes = [ip]
        L.hz_kernel_name.restype = C.c_char_p
        L.hz_noalloc_setup.argtypes = []
        L.hz_sum_fields_noalloc.argtypes = [vp, ip, C.c_longlong, ip, vp, vp]
        L.hz_strerror.argtypes = [ip]
        L.hz_strerror.restype = C.c_char_p
        _lib = L
    return _lib


def _chk(rc, where):
    if rc != 0:
        raise HzError(rc, where)


def _ptr(a):
    """Address of a numpy array (host) or a torch tensor (host or device)."""
    if isinstance(a, np.ndarray):
        return C.c_void_p(a.ctypes.data)
    return C.c_void_p(a.data_ptr())  # torch.Tensor


def noalloc_setup():
    """hz_noalloc_setup: device address of the fixed scratch array for the current device (no allocation)."""
    _chk(lib().hz_noalloc_setup(), "hz_noalloc_setup")


def sum_fields_noalloc(fields, nfields, ncell, out, stream=None):
    """hz_sum_fields_noalloc: out[f] = sum of plane f of `fields` (torch CUDA tensor, float32 or float64, nfields
    planes of ncell elements); `out` a torch CUDA tensor of nfields float64.  Asynchronous; allocates nothing."""
    import torch
    dt = HZ_F64 if fields.dtype == torch.float64 else HZ_F32
    s = getattr(stream, "cuda_stream", stream) if stream is not None else torch.cuda.current_stream().cuda_stream
    _chk(lib().hz_sum_fields_noalloc(_ptr(fields), int(nfields), int(ncell), dt, _ptr(out), C.c_void_p(s)),
         "hz_sum_fields_noalloc")
    return out


def fma_peak(dtype="f64"):
    """Measured FMA-pipe throughput in TFLOP/s (hz_fma_peak)."""
    t = C.c_double(0)
    _chk(lib().hz_fma_peak(HZ_F64 if dtype == "f64" else HZ_F32, C.byref(t)), "hz_fma_peak")
    return t.value


class Horizon:
    """One grid, one dtype.  Arrays in and out have shape (planes, nz, ny, nx), x fastest.

    Inputs may be numpy arrays (host) or torch tensors (host or CUDA) of the context dtype; other
    float arrays are converted.  `get_*` return numpy arrays unless `out=` (numpy or torch) is given.
    Device state lives in a torch.uint8 CUDA tensor (PyTorch is used for device memory and streams only).
    """

    def __init__(self, n, h, bc, dtype="f64", params=None, stream=None, use_torch_memory=True):
        import torch
        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the HORIZON update has no CPU fallback")
        self.n = tuple(int(x) for x in n)
        self.ncell = self.n[0] * self.n[1] * self.n[2]
        if dtype in ("f64", "float64", np.float64):
            self.dtype = HZ_F64
        elif dtype in ("f32", "float32", np.float32):
            self.dtype = HZ_F32
        elif dtype in ("f32h", "f32_f64", "mixed"):
            self.dtype = HZ_F32_F64      # fp32 storage and faces, fp64 flux difference / RK combine / con2prim
        else:
            raise ValueError(f"dtype must be 'f64', 'f32' or 'f32h', got {dtype!r}")
        self.np_dtype = np.float64 if self.dtype == HZ_F64 else np.float32
        self.grid = HzGrid(self.n[0], self.n[1], self.n[2], float(h[0]), float(h[1]), float(h[2]),
                           (C.c_int * 3)(*[int(b) for b in bc]))
        self.params = params if params is not None else HzParams.default()
        nbytes = C.c_size_t(0)
        _chk(L.hz_state_bytes_for(C.byref(self.grid), self.dtype, C.byref(self.params), C.byref(nbytes)),
             "hz_state_bytes_for")
        self.state_bytes = nbytes.value
        self._buf = None
        buf_ptr = None
        if use_torch_memory:
            self._buf = torch.empty(self.state_bytes + 256, dtype=torch.uint8, device="cuda")
            base = self._buf.data_ptr()
            buf_ptr = C.c_void_p((base + 255) // 256 * 256)
        h_ = C.c_void_p()
        _chk(L.hz_create(C.byref(self.grid), self.dtype, C.byref(self.params), buf_ptr, C.byref(h_)), "hz_create")
        self._h = h_
        if stream is not None:
            self.set_stream(stream)

    def close(self):
        if getattr(self, "_h", None):
            lib().hz_destroy(self._h)
            self._h = None
            self._buf = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- marshalling helpers ----
    def _in(self, a, planes):
        if isinstance(a, np.ndarray) or not hasattr(a, "data_ptr"):
            a = np.ascontiguousarray(np.asarray(a), dtype=self.np_dtype)
        else:
            import torch
            td = torch.float64 if self.dtype == HZ_F64 else torch.float32
            if a.dtype != td or not a.is_contiguous():
                a = a.to(td).contiguous()
        size = a.size if isinstance(a, np.ndarray) else a.numel()
        if size != planes * self.ncell:
            raise ValueError(f"expected {planes * self.ncell} values, got {size}")
        return a

    def _out(self, out, planes):
        if out is None:
            return np.empty((planes, self.n[2], self.n[1], self.n[0]), dtype=self.np_dtype)
        size = out.size if isinstance(out, np.ndarray) else out.numel()
        if size != planes * self.ncell:
            raise ValueError(f"expected {planes * self.ncell} values, got {size}")
        return out

    # ---- the C-ABI calls, same names ----
    def set_stream(self, stream):
        s = getattr(stream, "cuda_stream", stream)
        _chk(lib().hz_set_stream(self._h, C.c_void_p(s)), "hz_set_stream")

    def set_metric(self, alpha, beta3, gamma6):
        a, b, g = self._in(alpha, 1), self._in(beta3, 3), self._in(gamma6, 6)
        _chk(lib().hz_set_metric(self._h, _ptr(a), _ptr(b), _ptr(g)), "hz_set_metric")

    def set_primitives(self, prim8):
        a = self._in(prim8, 8)
        _chk(lib().hz_set_primitives(self._h, _ptr(a)), "hz_set_primitives")

    def step(self, dt, n):
        _chk(lib().hz_step(self._h, float(dt), int(n)), "hz_step")

    def substeps(self, dt, nsub):
        _chk(lib().hz_substeps(self._h, float(dt), int(nsub)), "hz_substeps")

    def get_primitives(self, out=None):
        out = self._out(out, 8)
        _chk(lib().hz_get_primitives(self._h, _ptr(out)), "hz_get_primitives")
        return out

    def get_psi(self, out=None):
        out = self._out(out, 1)
        _chk(lib().hz_get_psi(self._h, _ptr(out)), "hz_get_psi")
        return out[0] if isinstance(out, np.ndarray) else out

    def get_conserved(self, out=None):
        out = self._out(out, 9)
        _chk(lib().hz_get_conserved(self._h, _ptr(out)), "hz_get_conserved")
        return out

    def diagnostics(self):
        d = HzDiag()
        _chk(lib().hz_diagnostics(self._h, C.byref(d)), "hz_diagnostics")
        return d.asdict()

    def halo_bytes(self, which):
        n = C.c_size_t(0)
        _chk(lib().hz_halo_bytes(self._h, int(which), C.byref(n)), "hz_halo_bytes")
        return n.value

    def halo_pack(self, which, side, buf):
        """NG interior z planes next to `side` (0 low, 1 high) -> device buffer `buf` (torch CUDA tensor)."""
        _chk(lib().hz_halo_pack(self._h, int(which), int(side), _ptr(buf)), "hz_halo_pack")

    def halo_unpack(self, which, side, buf):
        """Device buffer `buf` -> ghost z planes of `side`."""
        _chk(lib().hz_halo_unpack(self._h, int(which), int(side), _ptr(buf)), "hz_halo_unpack")

    def prim_buffers(self):
        """(P0, P1, field_stride): device addresses of the two primitive sets (what a neighbour's peer_attach takes)."""
        p0, p1, fs = C.c_void_p(), C.c_void_p(), C.c_longlong(0)
        _chk(lib().hz_prim_buffers(self._h, C.byref(p0), C.byref(p1), C.byref(fs)), "hz_prim_buffers")
        return p0.value, p1.value, fs.value

    def peer_attach(self, side, p0, p1, field_stride, nz):
        """From now on every substep also stores the planes next to `side` into the neighbour's ghost planes."""
        _chk(lib().hz_peer_attach(self._h, int(side), C.c_void_p(p0), C.c_void_p(p1), int(field_stride), int(nz)),
             "hz_peer_attach")

    def peer_detach(self, side):
        _chk(lib().hz_peer_detach(self._h, int(side)), "hz_peer_detach")

    def launch_count(self):
        return lib().hz_launch_count(self._h)

    def profile(self, enable=True):
        _chk(lib().hz_profile(self._h, int(bool(enable))), "hz_profile")

    def profile_read(self):
        """{kernel name: (total ms, launches)} since the last read; synchronises."""
        ms = (C.c_double * HZ_NKERNELS)()
        cnt = (C.c_longlong * HZ_NKERNELS)()
        _chk(lib().hz_profile_read(self._h, ms, cnt), "hz_profile_read")
        return {lib().hz_kernel_name(k).decode(): (ms[k], cnt[k]) for k in range(HZ_NKERNELS)}

    @classmethod
    def from_workload(cls, w, dtype="f64", **kw):
        """Context for a workloads.Workload, with metric and primitives set."""
        par = HzParams.default(**w.params)
        hz = cls(w.n, w.h, w.bc, dtype=dtype, params=par, **kw)
        hz.set_metric(w.alpha, w.beta3, w.gamma6)
        hz.set_primitives(w.prim8)
        return hz

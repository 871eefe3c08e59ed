"""Thin ctypes binding of ``include/lbwp.h`` (argument marshalling only).

Every step of the path runs inside ``liblbwp.so`` (hand-written sm_100a kernels);
PyTorch is used here for device memory and streams only.  There is no CPU fallback:
if the library is missing or the device is not a B200-class GPU the calls raise.
Names mirror the C ABI: ``lbwp_init`` -> :class:`Lbwp`, ``lbwp_step`` -> ``step``,
``lbwp_moments`` -> ``moments`` / ``moments_host``.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "liblbwp.so")

LBWP_F32, LBWP_F64 = 0, 1
LBWP_MOMENTS, LBWP_POPULATIONS = 0, 1
KERNELS = {"auto": 0, "gather": 1, "march": 2, "tma": 3, "tma_split": 4}
EXPORTS = ["lbwp_state_bytes", "lbwp_num_moments", "lbwp_init", "lbwp_step", "lbwp_moments", "lbwp_diagnostics",
           "lbwp_diagnostics_static",
           "lbwp_halo_bytes", "lbwp_halo_pack", "lbwp_halo_unpack", "lbwp_set_moments", "lbwp_steps_done", "lbwp_launches_per_step", "lbwp_kernel_name",
           "lbwp_sync", "lbwp_destroy", "lbwp_last_error"]


class LbwpError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"lbwp error {code}: {text}")
        self.code = code


class Params(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_int32), ("lattice", ctypes.c_int32), ("dtype", ctypes.c_int32),
                ("ncomp", ctypes.c_int32), ("scheme", ctypes.c_int32), ("kernel", ctypes.c_int32),
                ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("device", ctypes.c_int32), ("tau", ctypes.c_double), ("A", ctypes.c_double),
                ("beta", ctypes.c_double), ("stream", ctypes.c_void_p), ("buf", ctypes.c_void_p * 2),
                ("A_h", ctypes.c_double), ("h_c", ctypes.c_double)]


class Diag(ctypes.Structure):
    _fields_ = [("mass", ctypes.c_double * 2), ("momentum", ctypes.c_double * 3), ("rho_mean_above", ctypes.c_double),
                ("rho_max", ctypes.c_double), ("count_above", ctypes.c_int64)]


_lib = None


def load():
    """dlopen liblbwp.so (must have been built: ``python -m paper_2301_01622_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise LbwpError(-4, f"{LIB_PATH} not built; run python -m paper_2301_01622_b200.build "
                            "(no CPU fallback exists)")
    lib = ctypes.CDLL(LIB_PATH)
    pp = ctypes.POINTER(Params)
    lib.lbwp_state_bytes.argtypes, lib.lbwp_state_bytes.restype = [pp], ctypes.c_size_t
    lib.lbwp_num_moments.argtypes, lib.lbwp_num_moments.restype = [pp], ctypes.c_int
    lib.lbwp_init.argtypes = [pp, ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_void_p)]
    lib.lbwp_step.argtypes = [ctypes.c_void_p, ctypes.c_int64]
    lib.lbwp_moments.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    lib.lbwp_set_moments.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    lib.lbwp_diagnostics.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.POINTER(ctypes.c_int32),
                                     ctypes.POINTER(Diag), ctypes.POINTER(ctypes.c_double)]
    lib.lbwp_diagnostics_static.argtypes = [ctypes.c_int] * 6 + [ctypes.c_void_p, ctypes.c_double, ctypes.c_int,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    lib.lbwp_halo_bytes.argtypes, lib.lbwp_halo_bytes.restype = [ctypes.c_void_p, ctypes.c_int], ctypes.c_size_t
    lib.lbwp_halo_pack.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
    lib.lbwp_halo_unpack.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
    lib.lbwp_steps_done.argtypes, lib.lbwp_steps_done.restype = [ctypes.c_void_p], ctypes.c_int64
    lib.lbwp_launches_per_step.argtypes = [ctypes.c_void_p]
    lib.lbwp_kernel_name.argtypes, lib.lbwp_kernel_name.restype = [ctypes.c_void_p], ctypes.c_char_p
    lib.lbwp_sync.argtypes = [ctypes.c_void_p]
    lib.lbwp_destroy.argtypes = [ctypes.c_void_p]
    lib.lbwp_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        raise LbwpError(rc, load().lbwp_last_error().decode())


def make_params(*, lattice, dtype, ncomp, shape, tau, A=0.0, beta=0.0, scheme="moments", kernel="auto",
                device=0, stream=0, buf=(None, None), A_h=0.0, h_c=4.0) -> Params:
    """shape = (nz, ny, nx) as in the external layout [M, nz, ny, nx]."""
    nz, ny, nx = shape
    p = Params()
    p.struct_size = ctypes.sizeof(Params)
    p.lattice, p.ncomp = int(lattice), int(ncomp)
    p.dtype = {"f32": LBWP_F32, "f64": LBWP_F64}[dtype]
    p.scheme = {"moments": LBWP_MOMENTS, "populations": LBWP_POPULATIONS}[scheme]
    p.kernel = KERNELS[kernel]
    p.nx, p.ny, p.nz = int(nx), int(ny), int(nz)
    p.device = int(device)
    p.tau, p.A, p.beta = float(tau), float(A), float(beta)
    p.A_h, p.h_c = float(A_h), float(h_c)
    p.stream = stream or None
    p.buf[0], p.buf[1] = buf
    return p


def state_bytes(params: Params) -> int:
    return int(load().lbwp_state_bytes(ctypes.byref(params)))


# limits of lbwp_diagnostics_static as include/lbwp.h states them
DIAG_STATIC_SCRATCH_BYTES = 42624
DIAG_STATIC_MAX_NODES = 1 << 31
DIAG_STATIC_MAX_PROBES = 4096
DIAG_STATIC_NOUT = 9


def diagnostics_static(moments, out, *, ncomp, threshold=0.5, probes=None, shape=None):
    """lbwp_diagnostics_static: the diagnostics of dense moments the CALLER holds, with no allocation in the library
    (its scratch is a static device array; calls that overlap on the GPU race on it).  Asynchronous on torch's current
    stream of the tensors' device.

    moments: contiguous CUDA tensor [M, nz, ny, nx], float32 or float64 (`shape` = (nz, ny, nx) overrides the tensor's
    own box, for callers that view a larger buffer); probes: None or a contiguous int32 CUDA tensor [n, 3] of
    (x, y, z); out: contiguous float64 CUDA tensor of at least 9 + n elements, written as include/lbwp.h lists."""
    import torch  # device pointers and the current stream only

    if not (moments.is_cuda and moments.is_contiguous() and moments.dtype in (torch.float32, torch.float64)):
        raise ValueError("moments must be a contiguous float32/float64 CUDA tensor")
    nz, ny, nx = (int(v) for v in (shape if shape is not None else moments.shape[1:]))
    n = 0 if probes is None else int(probes.shape[0])
    if n and not (probes.is_cuda and probes.is_contiguous() and probes.dtype == torch.int32 and probes.device == moments.device
                  and probes.dim() == 2 and probes.shape[1] == 3):
        raise ValueError("probes must be a contiguous int32 CUDA tensor [n, 3] on the moments' device")
    if not (out.is_cuda and out.is_contiguous() and out.dtype == torch.float64 and out.device == moments.device
            and out.numel() >= DIAG_STATIC_NOUT + n):
        raise ValueError("out must be a contiguous float64 CUDA tensor of at least 9 + nprobes elements on the moments' device")
    dev = moments.device.index if moments.device.index is not None else torch.cuda.current_device()
    _check(load().lbwp_diagnostics_static(dev, LBWP_F32 if moments.dtype == torch.float32 else LBWP_F64, int(ncomp), nx, ny, nz,
                                          ctypes.c_void_p(moments.data_ptr()), float(threshold), n,
                                          ctypes.c_void_p(probes.data_ptr()) if n else None, ctypes.c_void_p(out.data_ptr()),
                                          ctypes.c_void_p(torch.cuda.current_stream(moments.device).cuda_stream)))


class Lbwp:
    """One periodic box on one GPU (``lbwp_ctx``).  ``moments0``: numpy array (host) or torch
    CUDA tensor, external layout [M, nz, ny, nx] in the run's dtype."""

    def __init__(self, moments0, *, lattice=27, dtype="f32", ncomp=1, tau, A=0.0, beta=0.0,
                 scheme="moments", kernel="auto", device=0, use_torch_buffers=True, A_h=0.0, h_c=4.0):
        import torch  # device memory + stream only

        if not torch.cuda.is_available():
            raise LbwpError(-4, "no CUDA device: this library has no CPU fallback")
        self._torch = torch
        self.dtype = dtype
        self.np_dtype = np.float32 if dtype == "f32" else np.float64
        self.t_dtype = torch.float32 if dtype == "f32" else torch.float64
        self.M = 10 if ncomp == 1 else 11
        self.shape = tuple(int(s) for s in moments0.shape[1:])
        if moments0.shape[0] != self.M or len(moments0.shape) != 4:
            raise ValueError(f"moments must have shape [{self.M}, nz, ny, nx]")
        self.device = torch.device("cuda", device)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        p = make_params(lattice=lattice, dtype=dtype, ncomp=ncomp, shape=self.shape, tau=tau, A=A,
                        beta=beta, scheme=scheme, kernel=kernel, device=device, stream=stream, A_h=A_h, h_c=h_c)
        self.state_bytes = state_bytes(p)
        if self.state_bytes == 0:
            raise LbwpError(-1, "invalid parameters")
        self._bufs = None
        if use_torch_buffers:
            self._bufs = [torch.empty(self.state_bytes, dtype=torch.uint8, device=self.device) for _ in range(2)]
            p.buf[0], p.buf[1] = self._bufs[0].data_ptr(), self._bufs[1].data_ptr()
        self.params = p
        self._ctx = ctypes.c_void_p()
        ptr, on_dev, self._keep = self._marshal_in(moments0)
        _check(load().lbwp_init(ctypes.byref(p), ptr, on_dev, ctypes.byref(self._ctx)))
        self._keep = None

    def _marshal_in(self, m):
        torch = self._torch
        if isinstance(m, torch.Tensor):
            if m.dtype != self.t_dtype or not m.is_contiguous():
                raise ValueError("tensor must be contiguous and of the run's dtype")
            return ctypes.c_void_p(m.data_ptr()), int(m.is_cuda), m
        a = np.ascontiguousarray(m, dtype=self.np_dtype)
        return a.ctypes.data_as(ctypes.c_void_p), 0, a

    def step(self, n=1):
        """lbwp_step: enqueue n steps (asynchronous)."""
        _check(load().lbwp_step(self._ctx, int(n)))

    def set_moments(self, m):
        ptr, on_dev, keep = self._marshal_in(m)
        _check(load().lbwp_set_moments(self._ctx, ptr, on_dev))
        del keep

    def moments(self, out=None):
        """lbwp_moments into a torch CUDA tensor [M, nz, ny, nx] (synchronises)."""
        torch = self._torch
        if out is None:
            out = torch.empty((self.M, *self.shape), dtype=self.t_dtype, device=self.device)
        self._check_out(out)
        _check(load().lbwp_moments(self._ctx, ctypes.c_void_p(out.data_ptr()), int(out.is_cuda)))
        return out

    def _check_out(self, out):
        """The library writes M*nz*ny*nx elements of the run's dtype: refuse anything else (no silent overrun)."""
        shape = tuple(out.shape)
        if isinstance(out, np.ndarray):
            ok = out.dtype == self.np_dtype and out.flags["C_CONTIGUOUS"] and out.flags["WRITEABLE"]
        else:
            ok = out.dtype == self.t_dtype and out.is_contiguous()
            if out.is_cuda and out.device != self.device:
                ok = False
        if not ok or shape != (self.M, *self.shape):
            raise ValueError(f"out must be a contiguous [{self.M}, nz, ny, nx] = {(self.M, *self.shape)} array of {self.dtype}")

    def moments_host(self, out=None) -> np.ndarray:
        """lbwp_moments into a host numpy array (or a pinned torch CPU tensor passed as ``out``)."""
        if out is None:
            out = np.empty((self.M, *self.shape), dtype=self.np_dtype)
        self._check_out(out)
        if isinstance(out, np.ndarray):
            _check(load().lbwp_moments(self._ctx, out.ctypes.data_as(ctypes.c_void_p), 0))
        else:
            _check(load().lbwp_moments(self._ctx, ctypes.c_void_p(out.data_ptr()), 0))
        return out

    def diagnostics(self, threshold=0.5, probes=()):
        """lbwp_diagnostics: dict of the paper's diagnostics of the current state; probes = [(x, y, z), ...]."""
        n = len(probes)
        xyz = (ctypes.c_int32 * (3 * max(n, 1)))(*[int(v) for p in probes for v in p])
        rho = (ctypes.c_double * max(n, 1))()
        d = Diag()
        _check(load().lbwp_diagnostics(self._ctx, float(threshold), n, xyz if n else None, ctypes.byref(d), rho if n else None))
        return {"mass": [d.mass[0], d.mass[1]], "momentum": [d.momentum[0], d.momentum[1], d.momentum[2]],
                "rho_mean_above": d.rho_mean_above, "count_above": int(d.count_above), "rho_max": d.rho_max,
                "probe_rho": [rho[i] for i in range(n)]}

    def halo_bytes(self, nplanes) -> int:
        return int(load().lbwp_halo_bytes(self._ctx, int(nplanes)))

    def halo_pack(self, z0, nplanes, dst):
        """lbwp_halo_pack into a torch uint8 CUDA tensor of halo_bytes(nplanes) bytes (asynchronous)."""
        if dst.numel() * dst.element_size() < self.halo_bytes(nplanes) or not dst.is_cuda or not dst.is_contiguous():
            raise ValueError("dst must be a contiguous CUDA tensor of at least halo_bytes(nplanes) bytes")
        _check(load().lbwp_halo_pack(self._ctx, int(z0), int(nplanes), ctypes.c_void_p(dst.data_ptr())))

    def halo_unpack(self, z0, nplanes, src):
        if src.numel() * src.element_size() < self.halo_bytes(nplanes) or not src.is_cuda or not src.is_contiguous():
            raise ValueError("src must be a contiguous CUDA tensor of at least halo_bytes(nplanes) bytes")
        _check(load().lbwp_halo_unpack(self._ctx, int(z0), int(nplanes), ctypes.c_void_p(src.data_ptr())))

    def sync(self):
        _check(load().lbwp_sync(self._ctx))

    @property
    def steps_done(self) -> int:
        return int(load().lbwp_steps_done(self._ctx))

    @property
    def launches_per_step(self) -> int:
        return int(load().lbwp_launches_per_step(self._ctx))

    @property
    def kernel_name(self) -> str:
        return load().lbwp_kernel_name(self._ctx).decode()

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            load().lbwp_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()
            self._bufs = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

"""Thin ctypes binding over libpact.so (include/pact.h) — argument marshalling only.

Every step of the path (tau, Theta, W', their transposes) runs in the CUDA kernels behind the C
ABI; this module converts torch tensors to raw device pointers and checks return codes.  PyTorch
supplies device memory and the stream.  There is no CPU fallback: if the library is missing or no
CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_LIBPATH = _HERE / "libpact.so"

PACT_OK = 0
ERRORS = {-1: "PACT_EINVAL", -2: "PACT_ECFL", -3: "PACT_ERCV", -4: "PACT_EMATERIAL", -5: "PACT_ENOMEM",
          -6: "PACT_ECUDA", -7: "PACT_ENUMERIC"}
KERNEL_KINDS = ("fwd_vel", "fwd_str", "fwd_fused", "adj_a", "adj_b", "adj_fused", "recv", "other",
                "fwd_slab", "fwd_interior", "adj_slab", "adj_interior")       # PACT_K_* of include/pact.h

# every symbol include/pact.h declares (tests check that the library exports all of them)
SYMBOLS = ("pact_create", "pact_forward", "pact_adjoint", "pact_forward_host", "pact_adjoint_host",
           "pact_destroy", "pact_strerror", "pact_last_cuda_error", "pact_set_option", "pact_get_timing",
           "pact_device_bytes", "pact_get_info", "pact_pgd", "pact_power_iteration")


class PactParams(C.Structure):
    """Mirror of `pact_params` (include/pact.h)."""
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("h", C.c_double), ("dt", C.c_double),
                ("nt", C.c_int), ("npml", C.c_int), ("pml_R", C.c_double), ("pml_cref", C.c_double),
                ("pml_beta_max", C.c_double)]


class PactError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"{ERRORS.get(code, code)}: {text}")
        self.code = code


_lib = None


def lib():
    """Load libpact.so (raises if it has not been built: there is no fallback)."""
    global _lib
    if _lib is None:
        if not _LIBPATH.exists():
            raise RuntimeError(f"{_LIBPATH} is missing: run `python -m paper_1709_02733_b200.build`")
        L = C.CDLL(str(_LIBPATH))
        vp, ip, ll = C.c_void_p, C.c_int, C.c_longlong
        L.pact_create.restype = ip
        L.pact_create.argtypes = [C.POINTER(vp), C.POINTER(PactParams), vp, vp, vp, vp, vp, ip, vp]
        for name in ("pact_forward", "pact_adjoint", "pact_forward_host", "pact_adjoint_host"):
            getattr(L, name).restype = ip
            getattr(L, name).argtypes = [vp, vp, vp]
        L.pact_destroy.restype = None
        L.pact_destroy.argtypes = [vp]
        L.pact_strerror.restype = C.c_char_p
        L.pact_strerror.argtypes = [ip]
        L.pact_last_cuda_error.restype = C.c_char_p
        L.pact_last_cuda_error.argtypes = []
        L.pact_set_option.restype = ip
        L.pact_set_option.argtypes = [vp, C.c_char_p, ll]
        L.pact_get_timing.restype = ip
        L.pact_get_timing.argtypes = [vp, ip, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(ll)]
        L.pact_device_bytes.restype = ll
        L.pact_device_bytes.argtypes = [vp]
        L.pact_pgd.restype = ip
        L.pact_pgd.argtypes = [vp, vp, vp, C.c_double, ip, ip, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.pact_power_iteration.restype = ip
        L.pact_power_iteration.argtypes = [vp, vp, ip, C.POINTER(C.c_double)]
        L.pact_get_info.restype = ip
        L.pact_get_info.argtypes = [vp, C.c_char_p, C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _check(rc):
    if rc != PACT_OK:
        L = lib()
        text = L.pact_strerror(rc).decode()
        if rc == -6:
            text += " — " + L.pact_last_cuda_error().decode()
        raise PactError(rc, text)


def _dev_f32(t, shape, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float32 CUDA tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return C.c_void_p(t.data_ptr())


class Pact:
    """One `pact_ctx`: a medium, a receiver set and the operators H (forward) / H^T (adjoint).

    lam, mu, rho, alpha: float32 CUDA tensors [nz][ny][nx] (alpha may be None); rcv: [L][3] float64
    (numpy or CPU tensor), metres.  `prm` is any object with the fields of `pact_params`.
    """

    def __init__(self, prm, lam, mu, rho, alpha, rcv, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libpact needs a CUDA device (no CPU fallback)")
        L = lib()
        self.prm = prm
        self.shape = (prm.nz, prm.ny, prm.nx)
        self._p = PactParams(prm.nx, prm.ny, prm.nz, prm.h, prm.dt, prm.nt, prm.npml, prm.pml_R,
                             prm.pml_cref, prm.pml_beta_max)
        rcv = np.ascontiguousarray(np.asarray(rcv, dtype=np.float64)).reshape(-1, 3)
        self.L = int(rcv.shape[0])
        self.device = lam.device
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        ptrs = [_dev_f32(lam, self.shape, "lam"), _dev_f32(mu, self.shape, "mu"), _dev_f32(rho, self.shape, "rho"),
                _dev_f32(alpha, self.shape, "alpha") if alpha is not None else None]
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = L.pact_create(C.byref(h), C.byref(self._p), *ptrs, rcv.ctypes.data_as(C.c_void_p), self.L,
                               C.c_void_p(self.stream.cuda_stream))
        _check(rc)
        self._h = h

    @classmethod
    def from_problem(cls, prob, device="cuda:0", nt=None):
        """Upload a `synth.Problem` and create the context."""
        import torch
        from dataclasses import replace
        prm = prob.prm if nt is None else replace(prob.prm, nt=nt)
        dev = torch.device(device)
        up = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
        return cls(prm, up(prob.lam), up(prob.mu), up(prob.rho), up(prob.alpha) if prob.alpha is not None else None,
                   prob.rcv)

    def close(self):
        if getattr(self, "_h", None):
            lib().pact_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:       # interpreter shutdown: module globals may already be gone
            pass

    # ---- operators on device tensors (asynchronous on the context's stream)
    # Results are ordered on `self.stream` (the stream the context was created with) only.  Outputs the binding
    # allocates are allocated under that stream, inputs are recorded on it (so the caching allocator does not hand
    # their memory out while the library still reads it), and the caller's current stream is made to wait for the
    # library's work, so reading the result from the current stream is safe as well.
    def _enter(self, *inputs):
        import torch
        cur = torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)          # the inputs were produced on the caller's stream
            for t in inputs:
                t.record_stream(self.stream)
        return cur

    def _leave(self, cur):
        if cur != self.stream:
            cur.wait_stream(self.stream)

    def forward(self, p0, out=None):
        import torch
        cur = self._enter(p0)
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            if out is None:
                out = torch.empty((self.prm.nt, self.L), dtype=torch.float32, device=self.device)
            _check(lib().pact_forward(self._h, _dev_f32(p0, self.shape, "p0"),
                                      _dev_f32(out, (self.prm.nt, self.L), "data")))
        self._leave(cur)
        return out

    def adjoint(self, data, out=None):
        import torch
        cur = self._enter(data)
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            if out is None:
                out = torch.empty(self.shape, dtype=torch.float32, device=self.device)
            _check(lib().pact_adjoint(self._h, _dev_f32(data, (self.prm.nt, self.L), "data"),
                                      _dev_f32(out, self.shape, "image")))
        self._leave(cur)
        return out

    # ---- projected-gradient reconstruction (pact_pgd / pact_power_iteration): marshalling only
    def pgd(self, p, data, step, iters, nonneg=True):
        """In place on `p`: `iters` steps of p <- max(0, p - step H^T (H p - data)).  Returns
        (residual norms, update norms), one entry per iteration."""
        import torch
        cur = self._enter(p, data)
        res = (C.c_double * max(iters, 1))()
        upd = (C.c_double * max(iters, 1))()
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            _check(lib().pact_pgd(self._h, _dev_f32(p, self.shape, "p"), _dev_f32(data, (self.prm.nt, self.L), "data"),
                                  float(step), int(iters), int(bool(nonneg)), res, upd))
        self._leave(cur)
        return list(res)[:iters], list(upd)[:iters]

    def power_iteration(self, v, iters=8):
        """||H||^2 estimate; `v` (non-zero start vector) is overwritten by the normalised iterate."""
        import torch
        cur = self._enter(v)
        s2 = C.c_double()
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):
            _check(lib().pact_power_iteration(self._h, _dev_f32(v, self.shape, "v"), int(iters), C.byref(s2)))
        self._leave(cur)
        return s2.value

    # ---- operators on host buffers (copies inside; returns when the result is in host memory)
    def forward_host(self, p0_host, data_host):
        self._host_ok(p0_host, self.shape, "p0_host")
        self._host_ok(data_host, (self.prm.nt, self.L), "data_host")
        import torch
        with torch.cuda.device(self.device):
            _check(lib().pact_forward_host(self._h, C.c_void_p(p0_host.data_ptr()), C.c_void_p(data_host.data_ptr())))
        return data_host

    def adjoint_host(self, data_host, image_host):
        self._host_ok(data_host, (self.prm.nt, self.L), "data_host")
        self._host_ok(image_host, self.shape, "image_host")
        import torch
        with torch.cuda.device(self.device):
            _check(lib().pact_adjoint_host(self._h, C.c_void_p(data_host.data_ptr()), C.c_void_p(image_host.data_ptr())))
        return image_host

    @staticmethod
    def _host_ok(t, shape, name):
        import torch
        if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous float32 CPU tensor")
        if tuple(t.shape) != tuple(shape):
            raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")

    # ---- options / introspection
    def set_option(self, key, value):
        _check(lib().pact_set_option(self._h, key.encode(), int(value)))

    def timing(self, op):
        """(loop_ms, {kind: mean ms per launch}, {kind: launches}) of the last profiled forward
        (op = 0 or "forward") or adjoint (op = 1 or "adjoint") call."""
        op = {"forward": 0, "adjoint": 1}.get(op, op)
        loop = C.c_double()
        km = (C.c_double * len(KERNEL_KINDS))()
        ln = (C.c_longlong * len(KERNEL_KINDS))()
        _check(lib().pact_get_timing(self._h, int(op), C.byref(loop), km, ln))
        return loop.value, dict(zip(KERNEL_KINDS, km)), dict(zip(KERNEL_KINDS, ln))

    def info(self, key):
        v = C.c_double()
        _check(lib().pact_get_info(self._h, key.encode(), C.byref(v)))
        return v.value

    def device_bytes(self):
        return int(lib().pact_device_bytes(self._h))

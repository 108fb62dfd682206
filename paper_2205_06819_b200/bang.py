"""Python binding of libbang.so (include/bang.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory and streams.
There is no CPU fallback: if the shared library is missing or no CUDA device is present, calls fail loudly.
The function names mirror the C ABI: create / set_data / model_maps / model_fine / loglike (+ *_host).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbang.so")

BULGE, DISC1, DISC2, HALO = 1, 2, 4, 8
HALO_HERNQUIST, HALO_NFW = 0, 1
BULGE_HERNQUIST, BULGE_JAFFE = 0, 1
FP32, FP64 = 0, 1
PSF_FIELDS, PSF_FLUX = 0, 1
POTENTIAL_SELF, POTENTIAL_TOTAL = 0, 1
NTHETA = 17
NOALLOC_MAX_B = 65536            # include/bang.h: BANG_NOALLOC_MAX_B
OK, EINVAL, ENOMEM, ECUDA, ENODATA = 0, -1, -2, -3, -4

EXPORTS = ["bang_create", "bang_set_data", "bang_model_maps", "bang_model_fine", "bang_loglike", "bang_loglike_host",
           "bang_model_maps_host", "bang_loglike_noalloc", "bang_ns_walk", "bang_get_geometry", "bang_launch_count", "bang_probe_peaks", "bang_ml_from_colour", "bang_destroy", "bang_strerror",
           "bang_last_error"]


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("pix_arcsec", C.c_double), ("supersample", C.c_int),
                ("dist_mpc", C.c_double)]


class Psf(C.Structure):
    _fields_ = [("sigma_pix", C.c_double), ("trunc_nsigma", C.c_double)]


class Model(C.Structure):
    _fields_ = [("components", C.c_uint), ("bulge_profile", C.c_int), ("halo_profile", C.c_int),
                ("jeans_nodes", C.c_int), ("precision", C.c_int), ("psf_weighting", C.c_int), ("bulge_potential", C.c_int)]


class BangError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = code
        super().__init__(f"libbang error {code}: {detail}")


_lib = None


def lib():
    """Load libbang.so (built in-tree by paper_2205_06819_b200.build).  Raises if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not found: run `python -m paper_2205_06819_b200.build` "
                                    "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, ip, dp = C.c_void_p, C.c_int, C.c_double
        L.bang_create.argtypes = [C.POINTER(vp), C.POINTER(Grid), C.POINTER(Psf), C.POINTER(Model), ip, vp]
        L.bang_create.restype = ip
        L.bang_set_data.argtypes = [vp, vp, vp, vp]
        L.bang_set_data.restype = ip
        for name in ("bang_model_maps", "bang_model_fine", "bang_loglike", "bang_loglike_noalloc", "bang_loglike_host",
                     "bang_model_maps_host"):
            f = getattr(L, name)
            f.argtypes, f.restype = [vp, vp, ip, vp], ip
        L.bang_get_geometry.argtypes = [vp, C.POINTER(ip), C.POINTER(ip), C.POINTER(ip)]
        L.bang_get_geometry.restype = ip
        L.bang_launch_count.argtypes, L.bang_launch_count.restype = [vp], C.c_longlong
        L.bang_probe_peaks.argtypes, L.bang_probe_peaks.restype = [vp, C.POINTER(C.c_double)], ip
        L.bang_ml_from_colour.argtypes = [vp, vp, vp, vp, C.c_longlong, dp, dp, dp, vp, vp, ip, vp]
        L.bang_ml_from_colour.restype = ip
        L.bang_ns_walk.argtypes = [vp, ip, ip, vp, vp, vp, vp, vp, vp, vp, vp, ip, vp, vp, ip, C.c_ulonglong, vp]
        L.bang_ns_walk.restype = ip
        L.bang_destroy.argtypes, L.bang_destroy.restype = [vp], None
        L.bang_strerror.argtypes, L.bang_strerror.restype = [ip], C.c_char_p
        L.bang_last_error.argtypes, L.bang_last_error.restype = [vp], C.c_char_p
        _lib = L
    return _lib


class Context:
    """One bang_ctx: a grid, a PSF, a model variant and a precision, bound to a CUDA device and stream.

    Every kernel is enqueued on the context's stream (`ctx.stream`: the stream given at construction, else the device's
    current stream at that moment).  The temporaries this binding makes (theta uploaded from the host, output tensors)
    are allocated and filled under that same stream, so a caller working on another stream only has to order its own
    tensors against `ctx.stream` (torch.cuda.Stream.wait_stream).  The C entry points leave the calling thread's
    current CUDA device as they found it."""

    def __init__(self, cfg: dict, precision: str | None = None, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("bang.Context needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.cfg = dict(cfg)
        prec = precision or cfg.get("precision", "fp32")
        self.precision = prec
        self.dtype = torch.float64 if prec == "fp64" else torch.float32
        self.np_dtype = np.float64 if prec == "fp64" else np.float32
        self.device = torch.device("cuda", device)
        self.nx, self.ny, self.s = int(cfg["nx"]), int(cfg["ny"]), int(cfg["supersample"])
        g = Grid(self.nx, self.ny, float(cfg["pix_arcsec"]), self.s, float(cfg["dist_mpc"]))
        p = Psf(float(cfg["sigma_pix"]), float(cfg.get("trunc_nsigma", 3.0)))
        m = Model(int(cfg["components"]), int(cfg.get("bulge_profile", 0)), int(cfg.get("halo_profile", 0)), int(cfg["jeans_nodes"]),
                  FP64 if prec == "fp64" else FP32, int(cfg.get("psf_weighting", 0)), int(cfg.get("bulge_potential", 0)))
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = lib().bang_create(C.byref(h), C.byref(g), C.byref(p), C.byref(m), device,
                               C.c_void_p(self._stream.cuda_stream))
        if rc != OK:
            raise BangError(rc, lib().bang_strerror(rc).decode())
        self._h = h
        rk, nfx, nfy = C.c_int(), C.c_int(), C.c_int()
        lib().bang_get_geometry(self._h, C.byref(rk), C.byref(nfx), C.byref(nfy))
        self.r_k, self.nfx, self.nfy = rk.value, nfx.value, nfy.value

    # -- helpers
    def _check(self, rc):
        if rc != OK:
            raise BangError(rc, lib().bang_last_error(self._h).decode() or lib().bang_strerror(rc).decode())

    @property
    def stream(self):
        return self._stream

    def _on_stream(self):
        return self._torch.cuda.stream(self._stream)

    def _theta(self, theta):
        torch = self._torch
        t = torch.as_tensor(theta, dtype=torch.float64, device=self.device).reshape(-1, NTHETA).contiguous()
        return t

    def close(self):
        if getattr(self, "_h", None):
            lib().bang_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launches(self) -> int:
        return int(lib().bang_launch_count(self._h))

    # -- the ABI calls
    def set_data(self, data, err, mask):
        torch = self._torch
        d = torch.as_tensor(data, dtype=torch.float64, device=self.device).contiguous()
        e = torch.as_tensor(err, dtype=torch.float64, device=self.device).contiguous()
        m = torch.as_tensor(np.asarray(mask, dtype=np.uint8) if not torch.is_tensor(mask) else mask,
                            dtype=torch.uint8, device=self.device).contiguous()
        assert d.shape == (4, self.ny, self.nx) and e.shape == d.shape and m.shape == d.shape
        torch.cuda.current_stream(self.device).synchronize()         # the uploads above ran on the current stream
        self._check(lib().bang_set_data(self._h, d.data_ptr(), e.data_ptr(), m.data_ptr()))

    def model_maps(self, theta, out=None):
        """theta [B][17] (tensor on the device, or array-like) -> maps [B][4][ny][nx] device tensor (async)."""
        torch = self._torch
        with self._on_stream():
            t = self._theta(theta)
            B = t.shape[0]
            if out is None:
                out = torch.empty((B, 4, self.ny, self.nx), dtype=self.dtype, device=self.device)
            self._check(lib().bang_model_maps(self._h, t.data_ptr(), B, out.data_ptr()))
        return out

    def model_fine(self, theta):
        torch = self._torch
        with self._on_stream():
            t = self._theta(theta)
            B = t.shape[0]
            out = torch.empty((B, 4, self.nfy, self.nfx), dtype=self.dtype, device=self.device)
            self._check(lib().bang_model_fine(self._h, t.data_ptr(), B, out.data_ptr()))
        return out

    def loglike(self, theta, out=None):
        """theta [B][17] device tensor -> logL [B] float64 device tensor (async on the context's stream)."""
        torch = self._torch
        with self._on_stream():
            t = self._theta(theta)
            B = t.shape[0]
            if out is None:
                out = torch.empty((B,), dtype=torch.float64, device=self.device)
            self._check(lib().bang_loglike(self._h, t.data_ptr(), B, out.data_ptr()))
        return out

    def loglike_noalloc(self, theta, out):
        """bang_loglike_noalloc: theta [B][17] float64 device tensor, out [B] float64 device tensor, both made by the
        caller (this wrapper allocates nothing either); B <= NOALLOC_MAX_B.  Asynchronous on the context's stream."""
        torch = self._torch
        assert torch.is_tensor(theta) and theta.dtype == torch.float64 and theta.is_contiguous() and theta.device == self.device
        assert torch.is_tensor(out) and out.dtype == torch.float64 and out.is_contiguous() and out.device == self.device
        B = theta.shape[0]
        assert theta.shape == (B, NTHETA) and out.shape == (B,)
        with self._on_stream():
            self._check(lib().bang_loglike_noalloc(self._h, theta.data_ptr(), B, out.data_ptr()))
        return out

    def loglike_host(self, theta: np.ndarray, out: np.ndarray | None = None) -> np.ndarray:
        """HOST numpy theta [B][17] -> HOST numpy logL [B]; copies and synchronisation inside the call."""
        t = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, NTHETA)
        B = t.shape[0]
        if out is None:
            out = np.empty(B, dtype=np.float64)
        self._check(lib().bang_loglike_host(self._h, t.ctypes.data, B, out.ctypes.data))
        return out

    def ns_walk(self, u, logL, Lstar, group, chol, scale, free, lo, hi, theta0, steps: int, seed: int = 0) -> np.ndarray:
        """bang_ns_walk: advance the walkers u [K][d] (float64 device tensor, updated in place together with logL [K])
        by `steps` constrained Metropolis steps on the device.  Lstar [K] float64 and group [K] int32 device tensors;
        chol [G][d][d], scale [G], free [d], lo [d], hi [d], theta0 [17] host arrays.  Returns the accepted proposals per
        group (host int array); synchronises."""
        torch = self._torch
        K, d = u.shape
        chol = np.ascontiguousarray(chol, dtype=np.float64)
        G = chol.shape[0]
        assert chol.shape == (G, d, d) and u.dtype == torch.float64 and logL.dtype == torch.float64
        assert Lstar.dtype == torch.float64 and group.dtype == torch.int32 and u.is_contiguous()
        assert u.device == logL.device == Lstar.device == group.device == self.device
        scale = np.ascontiguousarray(scale, dtype=np.float64).reshape(G)
        free = np.ascontiguousarray(free, dtype=np.int32).reshape(d)
        lo = np.ascontiguousarray(lo, dtype=np.float64).reshape(d)
        hi = np.ascontiguousarray(hi, dtype=np.float64).reshape(d)
        theta0 = np.ascontiguousarray(theta0, dtype=np.float64).reshape(NTHETA)
        n_acc = np.zeros(G, dtype=np.int32)
        self._stream.wait_stream(torch.cuda.current_stream(self.device))    # the caller filled the tensors on its stream
        with self._on_stream():
            self._check(lib().bang_ns_walk(self._h, K, d, free.ctypes.data, lo.ctypes.data, hi.ctypes.data, theta0.ctypes.data,
                                           u.data_ptr(), logL.data_ptr(), Lstar.data_ptr(), group.data_ptr(), G,
                                           chol.ctypes.data, scale.ctypes.data, int(steps), int(seed) & (2**64 - 1),
                                           n_acc.ctypes.data))
        return n_acc

    def probe_peaks(self) -> dict:
        """Measured sustained instruction rates [thread-instr/s] of dependency-free FFMA, MUFU.EX2 and DFMA chains."""
        out = (C.c_double * 3)()
        self._check(lib().bang_probe_peaks(self._h, out))
        return {"fp32_fma": out[0], "mufu": out[1], "fp64_fma": out[2]}

    def model_maps_host(self, theta: np.ndarray) -> np.ndarray:
        t = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, NTHETA)
        B = t.shape[0]
        out = np.empty((B, 4, self.ny, self.nx), dtype=self.np_dtype)
        self._check(lib().bang_model_maps_host(self._h, t.ctypes.data, B, out.ctypes.data))
        return out


def ml_from_colour(m_beta, m_gamma, dm_beta, dm_gamma, a=-0.70, b=0.89, sigma_alpha=0.07, device=0):
    """eq. 20 with App. C's error model on the device: magnitude maps (and errors) -> (M/L, its error), float64 tensors."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bang.ml_from_colour needs a CUDA device (there is no CPU fallback)")
    dev = torch.device("cuda", device)
    x = [torch.as_tensor(v, dtype=torch.float64, device=dev).contiguous() for v in (m_beta, m_gamma, dm_beta, dm_gamma)]
    assert all(t.shape == x[0].shape for t in x)
    ml, err = torch.empty_like(x[0]), torch.empty_like(x[0])
    rc = lib().bang_ml_from_colour(x[0].data_ptr(), x[1].data_ptr(), x[2].data_ptr(), x[3].data_ptr(), x[0].numel(),
                                   float(a), float(b), float(sigma_alpha), ml.data_ptr(), err.data_ptr(), device,
                                   C.c_void_p(torch.cuda.current_stream(dev).cuda_stream))
    if rc != OK:
        raise BangError(rc, lib().bang_strerror(rc).decode())
    return ml, err

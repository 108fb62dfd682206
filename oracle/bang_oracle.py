"""ctypes wrapper around oracle/bang_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It holds no arithmetic of its own: every number comes from libbang_oracle.so.
The library is (re)built on demand with g++ (see build()).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bang_oracle.cpp")
_SO = os.path.join(_HERE, "libbang_oracle.so")

BULGE, DISC1, DISC2, HALO = 1, 2, 4, 8
HALO_HERNQUIST, HALO_NFW = 0, 1
BULGE_HERNQUIST, BULGE_JAFFE = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2 -fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _SO, "-lquadmath"]
        subprocess.run(cmd, check=True)
    return _SO


_lib = None
_d, _i, _u = C.c_double, C.c_int, C.c_uint
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_bp = np.ctypeslib.ndpointer(dtype=np.uint8, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        for name, args in {
            "bo_hernquist_X": [_d], "bo_sigma_tilde": [_d], "bo_I_tilde_closed": [_d],
            "bo_vr2_printed": [_d, _d, _d], "bo_T5": [_d], "bo_rho_vr2": [_d, _d, _d],
            "bo_Ib_quadrature": [_d, _d, _d, _i], "bo_freeman_F": [_d],
            "bo_vc2_hernquist": [_d, _d, _d], "bo_vc2_expdisc": [_d, _d, _d], "bo_nfw_mu": [_d],
            "bo_nfw_r200": [_d], "bo_vc2_nfw": [_d, _d, _d], "bo_hernquist_Sigma": [_d, _d, _d],
            "bo_G": [], "bo_kappa": [_d],
            "bo_jaffe_sigma_tilde": [_d], "bo_jaffe_I_tilde_closed": [_d], "bo_J3": [_d],
            "bo_rho_vr2_jaffe": [_d, _d, _d], "bo_vr2_jaffe_corrected": [_d, _d, _d], "bo_vc2_jaffe": [_d, _d, _d],
            "bo_Ib_quadrature_jaffe": [_d, _d, _d, _i],
            "bo_Ib_ext_quadrature": [_d, _d, _d, _i, _d, _d, _d, _d, _d, _d, _i, _u, _i],
            "bo_rho_bulge": [_d, _d, _d, _i],
        }.items():
            f = getattr(L, name)
            f.argtypes, f.restype = args, _d
        L.bo_set_threads.argtypes, L.bo_set_threads.restype = [_i], None
        L.bo_get_threads.argtypes, L.bo_get_threads.restype = [], _i
        L.bo_gauss_legendre.argtypes, L.bo_gauss_legendre.restype = [_i, _dp, _dp], None
        L.bo_psf_halfwidth.argtypes, L.bo_psf_halfwidth.restype = [_d, _i, _d], _i
        L.bo_psf_taps.argtypes, L.bo_psf_taps.restype = [_d, _i, _d, _dp], _i
        cfg = [_i, _i, _d, _i, _d, _d, _d, _u, _i, _i]   # nx ny pix s dist sigma trunc comps profiles NJ
        L.bo_model_fine.argtypes, L.bo_model_fine.restype = [_dp] + cfg + [_dp], _i
        L.bo_convolve_rebin.argtypes, L.bo_convolve_rebin.restype = [_dp, _i, _i, _i, _d, _d, _i, _dp], _i
        L.bo_model_maps.argtypes, L.bo_model_maps.restype = [_dp, _i] + cfg + [_dp], _i
        L.bo_loglike_of_maps.argtypes, L.bo_loglike_of_maps.restype = [_dp, _dp, _dp, _bp, _i, _i], _d
        L.bo_ml_from_colour.argtypes = [_dp, _dp, _dp, _dp, C.c_long, _d, _d, _d, _dp, _dp]
        L.bo_ml_from_colour.restype = None
        L.bo_loglike.argtypes = [_dp, _i] + cfg + [_dp, _dp, _bp, _dp, C.c_void_p]
        L.bo_loglike.restype = _i
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().bo_set_threads(int(n))


def get_threads() -> int:
    return int(lib().bo_get_threads())


def _cfg(cfg):
    """cfg: dict with nx ny pix_arcsec supersample dist_mpc sigma_pix trunc_nsigma components halo_profile
    [bulge_profile] jeans_nodes.  The switches travel in one int: halo | bulge << 8 | psf_weighting << 16 |
    bulge_potential << 24."""
    return (int(cfg["nx"]), int(cfg["ny"]), float(cfg["pix_arcsec"]), int(cfg["supersample"]),
            float(cfg["dist_mpc"]), float(cfg["sigma_pix"]), float(cfg.get("trunc_nsigma", 3.0)),
            int(cfg["components"]), int(cfg.get("halo_profile", 0)) | (int(cfg.get("bulge_profile", 0)) << 8) | (int(cfg.get("psf_weighting", 0)) << 16)
            | (int(cfg.get("bulge_potential", 0)) << 24),
            int(cfg["jeans_nodes"]))


def psf_halfwidth(cfg) -> int:
    return int(lib().bo_psf_halfwidth(float(cfg["sigma_pix"]), int(cfg["supersample"]),
                                      float(cfg.get("trunc_nsigma", 3.0))))


def psf_taps(sigma_pix: float, s: int, trunc: float = 3.0) -> np.ndarray:
    rk = lib().bo_psf_halfwidth(sigma_pix, s, trunc)
    g = np.zeros(2 * rk + 1)
    lib().bo_psf_taps(sigma_pix, s, trunc, g)
    return g


def gauss_legendre(n: int):
    x, w = np.zeros(n), np.zeros(n)
    lib().bo_gauss_legendre(n, x, w)
    return x, w


def model_fine(theta, cfg) -> np.ndarray:
    """Un-convolved fine maps [4][ny s + 2 r_k][nx s + 2 r_k] for one theta[17]."""
    theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(17)
    rk = psf_halfwidth(cfg)
    nfy = cfg["ny"] * cfg["supersample"] + 2 * rk
    nfx = cfg["nx"] * cfg["supersample"] + 2 * rk
    out = np.zeros((4, nfy, nfx))
    rc = lib().bo_model_fine(theta, *_cfg(cfg), out)
    if rc != 0:
        raise ValueError(f"bo_model_fine rc={rc}")
    return out


def convolve_rebin(fine, nx, ny, s, sigma_pix, trunc=3.0, psf_weighting=0) -> np.ndarray:
    fine = np.ascontiguousarray(fine, dtype=np.float64)
    out = np.zeros((4, ny, nx))
    rc = lib().bo_convolve_rebin(fine, nx, ny, s, sigma_pix, trunc, int(psf_weighting), out)
    if rc != 0:
        raise ValueError(f"bo_convolve_rebin rc={rc}")
    return out


def model_maps(theta, cfg) -> np.ndarray:
    """maps [B][4][ny][nx] for theta [B][17]."""
    theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 17)
    out = np.zeros((theta.shape[0], 4, cfg["ny"], cfg["nx"]))
    rc = lib().bo_model_maps(theta, theta.shape[0], *_cfg(cfg), out)
    if rc != 0:
        raise ValueError(f"bo_model_maps rc={rc}")
    return out


def loglike_of_maps(maps, data, err, mask) -> float:
    maps = np.ascontiguousarray(maps, dtype=np.float64)
    data = np.ascontiguousarray(data, dtype=np.float64)
    err = np.ascontiguousarray(err, dtype=np.float64)
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    ny, nx = maps.shape[-2:]
    return float(lib().bo_loglike_of_maps(maps, data, err, mask, nx, ny))


def loglike(theta, cfg, data, err, mask, return_maps: bool = False):
    theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 17)
    data = np.ascontiguousarray(data, dtype=np.float64)
    err = np.ascontiguousarray(err, dtype=np.float64)
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    B = theta.shape[0]
    out = np.zeros(B)
    maps = np.zeros((B, 4, cfg["ny"], cfg["nx"])) if return_maps else None
    mp = maps.ctypes.data_as(C.c_void_p) if return_maps else None
    rc = lib().bo_loglike(theta, B, *_cfg(cfg), data, err, mask, out, mp)
    if rc != 0:
        raise ValueError(f"bo_loglike rc={rc}")
    return (out, maps) if return_maps else out


def ml_from_colour(m_beta, m_gamma, dm_beta, dm_gamma, a=-0.70, b=0.89, sigma_alpha=0.07):
    """eq. 20 with App. C's error model (defaults: the paper's g-i / i-band constants)."""
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (m_beta, m_gamma, dm_beta, dm_gamma)]
    ml, err = np.empty_like(arrs[0]), np.empty_like(arrs[0])
    lib().bo_ml_from_colour(*[x.ravel() for x in arrs], arrs[0].size, a, b, sigma_alpha, ml.reshape(-1), err.reshape(-1))
    return ml, err

"""ctypes access to the CPU oracle (oracle/lsms_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_2308_16317_b200 and the CUDA
path never imports it.  All arithmetic is in lsms_oracle.cpp; this file only marshals
numpy arrays (column-major matrices are passed as flat interleaved (re,im) doubles).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lsms_oracle.cpp")
_LIB = os.path.join(_HERE, "liblsms_oracle.so")
_lib = None

_c_dp = ctypes.POINTER(ctypes.c_double)
_c_ip = ctypes.POINTER(ctypes.c_int32)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain -O2, OpenMP over batch items only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp",
                               "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        # LSMS_ORACLE_LIB: load another build of the same source (tests/test_oracle_sanitizers.py loads one compiled with
        # -fsanitize=address,undefined)
        _lib = ctypes.CDLL(os.environ.get("LSMS_ORACLE_LIB") or build())
        _lib.orc_tau00_full.restype = ctypes.c_int
        _lib.orc_tau00_schur.restype = ctypes.c_int
        _lib.orc_tau00_refined.restype = ctypes.c_int
        _lib.orc_inverse_gauss_jordan.restype = ctypes.c_int
        _lib.orc_tau00_batched.restype = ctypes.c_int
        _lib.orc_max_threads.restype = ctypes.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(_c_dp)


def _c2(z: complex) -> np.ndarray:
    return np.array([complex(z).real, complex(z).imag], dtype=np.float64)


def gaunt_quadrature(l, m, lp, mp, lpp, mpp) -> complex:
    out = np.zeros(2)
    lib().orc_gaunt_quadrature(int(l), int(m), int(lp), int(mp), int(lpp), int(mpp), _dp(out))
    return complex(out[0], out[1])


def gaunt_table(lmax: int) -> np.ndarray:
    kmax, nl2 = (lmax + 1) ** 2, (2 * lmax + 1) ** 2
    out = np.zeros((kmax, kmax, nl2))
    lib().orc_gaunt_table(int(lmax), _dp(out))
    return out


def ylm(lmax: int, v) -> np.ndarray:
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.zeros((lmax + 1) ** 2, dtype=np.complex128)
    lib().orc_ylm(int(lmax), _dp(v), _dp(out.view(np.float64)))
    return out


def hankel1(lmax: int, x: complex) -> np.ndarray:
    out = np.zeros(lmax + 1, dtype=np.complex128)
    lib().orc_hankel1(int(lmax), _dp(_c2(x)), _dp(out.view(np.float64)))
    return out


def g0_block(lmax: int, R, kappa: complex) -> np.ndarray:
    """g0_{LL'}(R; kappa) as a [kmax, kmax] array indexed [L, L']."""
    R = np.ascontiguousarray(R, dtype=np.float64)
    kmax = (lmax + 1) ** 2
    out = np.zeros(kmax * kmax, dtype=np.complex128)
    lib().orc_g0_block(int(lmax), _dp(R), _dp(_c2(kappa)), _dp(out.view(np.float64)))
    return out.reshape(kmax, kmax).T.copy()      # stored L + kmax*L'


def tinv(delta: complex, kappa: complex) -> complex:
    out = np.zeros(2)
    lib().orc_tinv(_dp(_c2(delta)), _dp(_c2(kappa)), _dp(out))
    return complex(out[0], out[1])


def assemble_M(n_sites, lmax, canted, site_pos, species, delta, moment, z) -> np.ndarray:
    """KKR matrix of one item as a numpy [n, n] array indexed [row, col]."""
    k = (lmax + 1) ** 2 * (2 if canted else 1)
    n = n_sites * k
    site_pos = np.ascontiguousarray(site_pos, dtype=np.float64)
    species = np.ascontiguousarray(species, dtype=np.int32)
    delta = np.ascontiguousarray(delta, dtype=np.complex128)
    moment = np.ascontiguousarray(moment, dtype=np.float64)
    M = np.zeros(n * n, dtype=np.complex128)
    lib().orc_assemble_M(int(n_sites), int(lmax), int(bool(canted)), _dp(site_pos),
                         species.ctypes.data_as(_c_ip), _dp(delta.view(np.float64)), _dp(moment),
                         _dp(_c2(z)), _dp(M.view(np.float64)))
    return M.reshape(n, n).T           # column-major storage -> [row, col] view


def _colmajor(M: np.ndarray) -> np.ndarray:
    """flat column-major copy of a [row, col] array"""
    return np.ascontiguousarray(np.asarray(M, dtype=np.complex128).T).ravel()


def tau00_full(M: np.ndarray, k: int, precision: str = "double", want_X: bool = False):
    """Textbook route: X = M^{-1} E_last via Gaussian elimination with unrestricted partial
    pivoting on [M | E]; tau00 = last k rows of X."""
    n = M.shape[0]
    flat = _colmajor(M)
    tau = np.zeros(k * k, dtype=np.complex128)
    X = np.zeros(n * k, dtype=np.complex128) if want_X else None
    info = lib().orc_tau00_full(n, int(k), _dp(flat.view(np.float64)), 1 if precision == "long double" else 0,
                                _dp(tau.view(np.float64)), _dp(X.view(np.float64)) if want_X else None)
    if info:
        raise np.linalg.LinAlgError(f"zero pivot at step {info}")
    tau = tau.reshape(k, k).T.copy()
    return (tau, X.reshape(k, n).T.copy()) if want_X else tau


def tau00_schur(M: np.ndarray, k: int) -> np.ndarray:
    n = M.shape[0]
    flat = _colmajor(M)
    tau = np.zeros(k * k, dtype=np.complex128)
    info = lib().orc_tau00_schur(n, int(k), _dp(flat.view(np.float64)), _dp(tau.view(np.float64)))
    if info:
        raise np.linalg.LinAlgError(f"zero pivot at step {info}")
    return tau.reshape(k, k).T.copy()


def tau00_refined(M: np.ndarray, k: int, n_refine: int = 2, want_X: bool = False):
    n = M.shape[0]
    flat = _colmajor(M)
    tau = np.zeros(k * k, dtype=np.complex128)
    X = np.zeros(n * k, dtype=np.complex128) if want_X else None
    info = lib().orc_tau00_refined(n, int(k), _dp(flat.view(np.float64)), int(n_refine),
                                   _dp(tau.view(np.float64)), _dp(X.view(np.float64)) if want_X else None)
    if info:
        raise np.linalg.LinAlgError(f"zero pivot at step {info}")
    tau = tau.reshape(k, k).T.copy()
    return (tau, X.reshape(k, n).T.copy()) if want_X else tau


def inverse_gauss_jordan(M: np.ndarray) -> np.ndarray:
    n = M.shape[0]
    flat = _colmajor(M)
    inv = np.zeros(n * n, dtype=np.complex128)
    info = lib().orc_inverse_gauss_jordan(n, _dp(flat.view(np.float64)), _dp(inv.view(np.float64)))
    if info:
        raise np.linalg.LinAlgError(f"zero pivot at step {info}")
    return inv.reshape(n, n).T.copy()


def tau00_batched(batch, mode: str = "double") -> tuple[np.ndarray, np.ndarray]:
    """Whole path (assembly + textbook solve) for a synth_liz.LizBatch-like object;
    OpenMP over items.  Returns (tau [batch,k,k] indexed [b,row,col], info [batch])."""
    cfg = batch.cfg
    B, k = batch.batch, cfg.k
    site_pos = np.ascontiguousarray(batch.site_pos, dtype=np.float64)
    species = np.ascontiguousarray(batch.species, dtype=np.int32)
    delta = np.ascontiguousarray(batch.delta, dtype=np.complex128)
    moment = np.ascontiguousarray(batch.moment_dir, dtype=np.float64)
    z = np.ascontiguousarray(batch.z, dtype=np.complex128)
    tau = np.zeros((B, k * k), dtype=np.complex128)
    info = np.zeros(B, dtype=np.int32)
    m = {"double": 0, "long double": 1, "schur": 2}[mode]
    lib().orc_tau00_batched(B, cfg.n_sites, cfg.lmax, int(cfg.spin_canted), _dp(site_pos),
                            species.ctypes.data_as(_c_ip), _dp(delta.view(np.float64)), _dp(moment),
                            _dp(z.view(np.float64)), m, _dp(tau.view(np.float64)),
                            info.ctypes.data_as(_c_ip))
    return tau.reshape(B, k, k).transpose(0, 2, 1).copy(), info


def max_threads() -> int:
    return int(lib().orc_max_threads())


def contour_sum(tau: np.ndarray, w: np.ndarray) -> np.ndarray:
    """out[a] = sum_q w[q] tau[a, q]  (the tau part of eq. (2)/(3)).
    tau complex128 [n_atoms, n_e, ...], w complex128 [n_e]."""
    tau = np.ascontiguousarray(tau, dtype=np.complex128)
    w = np.ascontiguousarray(w, dtype=np.complex128)
    na, ne = tau.shape[0], tau.shape[1]
    kk = int(np.prod(tau.shape[2:]))
    out = np.zeros((na,) + tau.shape[2:], dtype=np.complex128)
    lib().orc_contour_sum(na, ne, kk, _dp(tau.view(np.float64)), _dp(w.view(np.float64)), _dp(out.view(np.float64)))
    return out


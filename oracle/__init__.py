"""ctypes front-end of the fp64 CPU oracle (oracle/gwmf_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports the CUDA
binding, and the CUDA binding never imports it.

The C file is compiled on first use with the system gcc (``oracle/build.py``); all arithmetic
lives in C, this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gwmf_oracle.c")
_LIB = os.path.join(_HERE, "libgwmf_oracle.so")


def build(force: bool = False) -> str:
    """Compile gwmf_oracle.c -> libgwmf_oracle.so (gcc -O2 -fopenmp; strict IEEE, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
    return _LIB


_lib = None
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_lp = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_t_sun.restype = C.c_double
        L.orc_dft_naive.argtypes = [_dp, _dp, _dp, _dp, C.c_long, C.c_int]
        L.orc_fft_radix2.argtypes = [_dp, _dp, C.c_long, C.c_int]
        L.orc_psd_eq2.argtypes = [C.c_double]
        L.orc_psd_eq2.restype = C.c_double
        L.orc_f_isco.argtypes = [C.c_double, C.c_double]
        L.orc_f_isco.restype = C.c_double
        L.orc_k_high.argtypes = [C.c_double, C.c_double, C.c_long, C.c_double]
        L.orc_k_high.restype = C.c_long
        L.orc_k_low.argtypes = [C.c_long, C.c_double, C.c_double]
        L.orc_k_low.restype = C.c_long
        L.orc_phase.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_amplitude.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_amplitude.restype = C.c_double
        L.orc_phase.restype = C.c_double
        L.orc_template.argtypes = [C.c_double, C.c_double, C.c_long, C.c_double, C.c_double, _dp, _dp]
        L.orc_power_table.argtypes = [_dp, C.c_long, C.c_double, C.c_double, _dp]
        L.orc_sigma_edges.argtypes = [_dp, C.c_long, C.c_double, C.c_double, C.c_long, C.c_int,
                                      C.POINTER(C.c_double), _lp]
        L.orc_data_spectrum.argtypes = [_dp, C.c_long, _dp, _dp]
        L.orc_filter_template.argtypes = [_dp, _dp, _dp, _dp, C.c_long, C.c_double, C.c_double,
                                          C.c_double, C.c_double, C.c_int, _dp, _dp,
                                          C.POINTER(C.c_double), _lp, C.c_void_p, C.c_void_p]
        L.orc_filter_template_bruteforce.argtypes = [_dp, _dp, C.c_long, C.c_double, C.c_double,
                                                     C.c_double, C.c_double, C.c_int, _dp, _dp,
                                                     C.POINTER(C.c_double), _lp]
        L.orc_window_maxima.argtypes = [_dp, _dp, C.c_long, C.c_long, C.c_double, _lp, _dp, _dp, _dp]
        L.orc_window_maxima.restype = C.c_long
        L.orc_filter_bank.argtypes = [_dp, _dp, C.c_long, C.c_double, C.c_double, _dp, _dp, C.c_long,
                                      C.c_int, C.c_long, C.c_double, _dp, _lp, _lp, _dp, _dp, _dp,
                                      _ip, C.c_long, C.c_void_p, C.c_void_p, C.c_int]
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ------------------------------------------------------------------ transforms
def fft(x: np.ndarray, sign: int) -> np.ndarray:
    """Unnormalised radix-2 DFT, X[k] = sum_j x[j] e^{sign 2 pi i jk/n}."""
    x = np.asarray(x, dtype=np.complex128)
    re, im = _f64(x.real).copy(), _f64(x.imag).copy()
    rc = lib().orc_fft_radix2(re, im, len(x), sign)
    if rc:
        raise ValueError(f"orc_fft_radix2 -> {rc}")
    return re + 1j * im


def dft_naive(x: np.ndarray, sign: int) -> np.ndarray:
    x = np.asarray(x, dtype=np.complex128)
    yr, yi = np.empty(len(x)), np.empty(len(x))
    lib().orc_dft_naive(_f64(x.real), _f64(x.imag), yr, yi, len(x), sign)
    return yr + 1j * yi


# ------------------------------------------------------------------ scalar pieces
def t_sun() -> float:
    return lib().orc_t_sun()


def psd_eq2(f: float) -> float:
    return lib().orc_psd_eq2(float(f))


def f_isco(m1, m2) -> float:
    return lib().orc_f_isco(float(m1), float(m2))


def k_low(n, fs=4096.0, f_low=40.0) -> int:
    return lib().orc_k_low(int(n), float(fs), float(f_low))


def k_high(m1, m2, n, fs=4096.0) -> int:
    return lib().orc_k_high(float(m1), float(m2), int(n), float(fs))


def phase(m1, m2, f) -> float:
    return lib().orc_phase(float(m1), float(m2), float(f))


def amplitude(m1, m2, d_eff_mpc=1.0) -> float:
    """Physical amplitude constant of the template for a source at d_eff_mpc megaparsecs (O10)."""
    return lib().orc_amplitude(float(m1), float(m2), float(d_eff_mpc))


def template(m1, m2, n, fs=4096.0, f_low=40.0) -> np.ndarray:
    hr, hi = np.empty(n // 2), np.empty(n // 2)
    lib().orc_template(float(m1), float(m2), int(n), float(fs), float(f_low), hr, hi)
    return hr + 1j * hi


def power_table(Sn, n, fs=4096.0, f_low=40.0) -> np.ndarray:
    c = np.empty(n // 2)
    lib().orc_power_table(_f64(Sn), int(n), float(fs), float(f_low), c)
    return c


def sigma_edges(Ctab, n, kh, p, fs=4096.0, f_low=40.0):
    sig = C.c_double(0.0)
    edges = np.zeros(p + 1, dtype=np.int64)
    rc = lib().orc_sigma_edges(_f64(Ctab), int(n), float(fs), float(f_low), int(kh), int(p),
                               C.byref(sig), edges)
    if rc:
        raise ValueError(f"orc_sigma_edges -> {rc}")
    return sig.value, edges


def data_spectrum(s) -> np.ndarray:
    s = _f64(s)
    n = len(s)
    dr, di = np.empty(n // 2 + 1), np.empty(n // 2 + 1)
    rc = lib().orc_data_spectrum(s, n, dr, di)
    if rc:
        raise ValueError(f"orc_data_spectrum -> {rc}")
    return dr + 1j * di


# ------------------------------------------------------------------ one template
def filter_template(s, Sn, m1, m2, p, fs=4096.0, f_low=40.0, bands=False, D=None, Ctab=None):
    """rho[n], chisq[n], sigma, edges[p+1] (and the p band series if bands=True)."""
    s = _f64(s)
    Sn = _f64(Sn)
    n = len(s)
    if D is None:
        D = data_spectrum(s)
    if Ctab is None:
        Ctab = power_table(Sn, n, fs, f_low)
    rho, chi = np.empty(n), np.empty(n)
    sig = C.c_double(0.0)
    edges = np.zeros(p + 1, dtype=np.int64)
    zr = zi = None
    zrp = zip_ = None
    if bands:
        zr, zi = np.empty((p, n)), np.empty((p, n))
        zrp, zip_ = zr.ctypes.data_as(C.c_void_p), zi.ctypes.data_as(C.c_void_p)
    rc = lib().orc_filter_template(_f64(D.real), _f64(D.imag), Sn, _f64(Ctab), n, float(fs), float(f_low),
                                   float(m1), float(m2), int(p), rho, chi, C.byref(sig), edges, zrp, zip_)
    if rc:
        raise ValueError(f"orc_filter_template -> {rc}")
    if bands:
        return rho, chi, sig.value, edges, zr + 1j * zi
    return rho, chi, sig.value, edges


def filter_template_bruteforce(s, Sn, m1, m2, p, fs=4096.0, f_low=40.0):
    s = _f64(s)
    n = len(s)
    rho, chi = np.empty(n), np.empty(n)
    sig = C.c_double(0.0)
    edges = np.zeros(p + 1, dtype=np.int64)
    rc = lib().orc_filter_template_bruteforce(s, _f64(Sn), n, float(fs), float(f_low), float(m1), float(m2),
                                              int(p), rho, chi, C.byref(sig), edges)
    if rc:
        raise ValueError(f"orc_filter_template_bruteforce -> {rc}")
    return rho, chi, sig.value, edges


def window_maxima(rho, chisq, W, thresh):
    rho, chisq = _f64(rho), _f64(chisq)
    n = len(rho)
    nw = n // W
    bj = np.zeros(nw, dtype=np.int64)
    br, bc, ru = np.empty(nw), np.empty(nw), np.empty(nw)
    cnt = lib().orc_window_maxima(rho, chisq, n, int(W), float(thresh), bj, br, bc, ru)
    return cnt, bj, br, bc, ru


# ------------------------------------------------------------------ whole bank
def filter_bank(s, Sn, masses, p, W, thresh, fs=4096.0, f_low=40.0, keep=-1, n_threads=None):
    """All templates of `masses` against one segment.

    Returns dict(sigma[T], edges[T,p+1], best_j[T,nw], best_rho, best_chisq, runner_up, status[T],
    rho_keep, chisq_keep).  Triggers are the (t, w) cells with best_rho > thresh.
    """
    s, Sn = _f64(s), _f64(Sn)
    n = len(s)
    T = len(masses)
    nw = n // W
    m1 = _f64([m[0] for m in masses])
    m2 = _f64([m[1] for m in masses])
    out = dict(sigma=np.zeros(T), edges=np.zeros((T, p + 1), dtype=np.int64),
               best_j=np.zeros((T, nw), dtype=np.int64), best_rho=np.zeros((T, nw)),
               best_chisq=np.zeros((T, nw)), runner_up=np.zeros((T, nw)),
               status=np.zeros(T, dtype=np.int32))
    rk = ck = None
    rkp = ckp = None
    if 0 <= keep < T:
        rk, ck = np.empty(n), np.empty(n)
        rkp, ckp = rk.ctypes.data_as(C.c_void_p), ck.ctypes.data_as(C.c_void_p)
    if n_threads is None:
        n_threads = os.cpu_count() or 1
    rc = lib().orc_filter_bank(s, Sn, n, float(fs), float(f_low), m1, m2, T, int(p), int(W), float(thresh),
                               out["sigma"], out["edges"].reshape(-1), out["best_j"].reshape(-1),
                               out["best_rho"].reshape(-1), out["best_chisq"].reshape(-1),
                               out["runner_up"].reshape(-1), out["status"], int(keep), rkp, ckp,
                               int(n_threads))
    if rc:
        raise ValueError(f"orc_filter_bank -> {rc}")
    out["rho_keep"], out["chisq_keep"] = rk, ck
    out["threads"] = n_threads
    return out


def triggers(bank_out, thresh):
    """(template, sample, rho, chisq) rows sorted by (template, window) -- O9."""
    rows = []
    T, nw = bank_out["best_rho"].shape
    for t in range(T):
        for w in range(nw):
            if bank_out["best_rho"][t, w] > thresh:
                rows.append((t, int(bank_out["best_j"][t, w]), float(bank_out["best_rho"][t, w]),
                             float(bank_out["best_chisq"][t, w])))
    return rows

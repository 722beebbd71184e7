"""CPU oracle for the Pulscan boxcar-search hot path — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes wrapper over ``pulscan_oracle.c`` (plain C, double precision, written from PAPER.md; see that file's
header for the citations and the pins).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2406_15186_b200`` and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "pulscan_oracle.c"
# ORACLE_SANITIZE=1 in the environment: build and load an AddressSanitizer + UBSan copy instead (run the CPU tests with
# LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0; DESIGN.md §7 records the last such run)
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
_LIB = _HERE / ("liboracle_san.so" if _SANITIZE else "liboracle.so")

CANDIDATE_DTYPE = np.dtype(
    [("spectrum", "<i4"), ("bin", "<i4"), ("width", "<i4"), ("numharm", "<i4"), ("power", "<f8"), ("sigma", "<f8"),
     ("lnp", "<f8")]
)


def build(force: bool = False) -> Path:
    """Compile the C oracle with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        san = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SANITIZE else []
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-D_GNU_SOURCE", *san, "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(str(build()))
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_fp = ctypes.POINTER(ctypes.c_float)
        c_lp = ctypes.POINTER(ctypes.c_int64)
        lib.orc_median.restype = ctypes.c_double
        lib.orc_median.argtypes = [c_dp, ctypes.c_int64, c_dp]
        lib.orc_normalise_block.restype = ctypes.c_double
        lib.orc_normalise_block.argtypes = [c_dp, ctypes.c_int64, c_dp, c_dp, c_dp]
        lib.orc_normalise_power.restype = None
        lib.orc_normalise_power.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, c_dp]
        lib.orc_boxcar_sums.restype = None
        lib.orc_boxcar_sums.argtypes = [c_dp, ctypes.c_int64, ctypes.c_int32, c_dp]
        lib.orc_block_maxima.restype = None
        lib.orc_block_maxima.argtypes = [c_dp, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64, c_dp, c_dp, c_lp]
        lib.orc_ln_q.restype = ctypes.c_double
        lib.orc_ln_q.argtypes = [ctypes.c_int32, ctypes.c_double]
        lib.orc_ln_sf.restype = ctypes.c_double
        lib.orc_ln_sf.argtypes = [ctypes.c_double]
        lib.orc_sigma_from_lnp.restype = ctypes.c_double
        lib.orc_sigma_from_lnp.argtypes = [ctypes.c_double]
        lib.orc_power_threshold.restype = ctypes.c_double
        lib.orc_power_threshold.argtypes = [ctypes.c_int32, ctypes.c_double]
        lib.orc_width_searched.restype = ctypes.c_int32
        lib.orc_width_searched.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32]
        lib.orc_search_sampled.restype = ctypes.c_int64
        lib.orc_search_sampled.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                           ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int32, ctypes.c_int32,
                                           ctypes.c_void_p, ctypes.c_int64]
        lib.orc_search_ex.restype = ctypes.c_int64
        lib.orc_search_ex.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                      ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int32, ctypes.c_int32,
                                      ctypes.c_int32, ctypes.c_void_p, ctypes.c_int64]
        lib.orc_harmonic_sum.restype = ctypes.c_int64
        lib.orc_harmonic_sum.argtypes = [c_dp, ctypes.c_int64, ctypes.c_int32, c_dp]
        lib.orc_search_harmonics.restype = ctypes.c_int64
        lib.orc_search_harmonics.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                             ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int32, ctypes.c_int32,
                                             ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int64]
        lib.orc_median_of_medians.restype = ctypes.c_double
        lib.orc_median_of_medians.argtypes = [c_dp, ctypes.c_int64]
        lib.orc_normalise_power_mom.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, c_dp]
        lib.orc_search_general.restype = ctypes.c_int64
        lib.orc_search_general.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                           ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int32, ctypes.c_int32,
                                           ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int64]
        lib.orc_search_opts.restype = ctypes.c_int64
        lib.orc_search_opts.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                        ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int32, ctypes.c_int32,
                                        ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p,
                                        ctypes.c_int64]
        lib.orc_search_all.restype = ctypes.c_int64
        lib.orc_search_all.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                       ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int32, ctypes.c_int32,
                                       ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                       ctypes.c_void_p, ctypes.c_int64]
        lib.orc_power_to_logp.restype = ctypes.c_double
        lib.orc_power_to_logp.argtypes = [ctypes.c_double, ctypes.c_double]
        lib.orc_search.restype = ctypes.c_int64
        lib.orc_search.argtypes = [c_fp, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64,
                                   ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_void_p, ctypes.c_int64]
        lib.orc_num_threads.restype = ctypes.c_int
        lib.orc_kappa.restype = ctypes.c_double
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def kappa() -> float:
    """1/Φ⁻¹(3/4), the MAD → standard-deviation factor."""
    return float(_load().orc_kappa())


def num_threads() -> int:
    return int(_load().orc_num_threads())


def median(v) -> float:
    v = np.ascontiguousarray(v, dtype=np.float64)
    scratch = np.empty_like(v)
    return float(_load().orc_median(_dp(v), v.size, _dp(scratch)))


def normalise_block(v):
    """(v − median)/(κ·MAD) of one real block (Eq. 8).  Returns (normalised, median, scale)."""
    out = np.array(v, dtype=np.float64, copy=True)
    scratch = np.empty_like(out)
    dev = np.empty_like(out)
    scale = ctypes.c_double()
    med = _load().orc_normalise_block(_dp(out), out.size, _dp(scratch), _dp(dev), ctypes.byref(scale))
    return out, float(med), float(scale.value)


def _as_interleaved(spectrum) -> np.ndarray:
    s = np.ascontiguousarray(spectrum, dtype=np.complex64)
    return s.view(np.float32)


def normalise_power(spectrum, norm_block: int) -> np.ndarray:
    """Steps 1-3: per-block, per-component median/MAD normalisation, then P = |X'|²/2 (float64, one spectrum)."""
    f = _as_interleaved(spectrum).reshape(-1)
    n = f.size // 2
    P = np.empty(n, dtype=np.float64)
    _load().orc_normalise_power(f.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), n, int(norm_block), _dp(P))
    return P


def boxcar_sums(P, zmax: int) -> np.ndarray:
    """All S(i,w) by the paper's recursion; returns [zmax, n] with NaN where the window does not exist."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    out = np.empty((int(zmax), P.size), dtype=np.float64)
    _load().orc_boxcar_sums(_dp(P), P.size, int(zmax), _dp(out))
    return out


def block_maxima(P, zmax: int, block_width: int):
    """M(c,w), I(c,w) for every candidate block: arrays [n_blocks, zmax]; −1 where no window exists."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    n, C = P.size, int(block_width)
    nblk = (n + C - 1) // C
    M = np.empty((nblk, zmax), dtype=np.float64)
    I = np.empty((nblk, zmax), dtype=np.int64)
    sums = np.empty(C, dtype=np.float64)
    lib = _load()
    for c in range(nblk):
        lib.orc_block_maxima(_dp(P), n, int(zmax), C, c, _dp(sums), _dp(M[c]),
                             I[c].ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
    return M, I


def ln_q(w: int, S: float) -> float:
    """ln of the χ²(2w) survival function at 2S (Eq. 9)."""
    return float(_load().orc_ln_q(int(w), float(S)))


def power_to_logp(power: float, dof: float) -> float:
    """Alg. 3: the paper's polynomial approximation of ln p, in the paper's units (χ² power, d.o.f.)."""
    return float(_load().orc_power_to_logp(float(power), float(dof)))


def ln_sf(x: float) -> float:
    return float(_load().orc_ln_sf(float(x)))


def sigma_from_lnp(lnp: float) -> float:
    return float(_load().orc_sigma_from_lnp(float(lnp)))


def power_threshold(w: int, sigma_threshold: float, n_trials: float = 1.0) -> float:
    """T_w: the power at which a width-w boxcar reaches the σ threshold."""
    return float(_load().orc_power_threshold(int(w), ln_sf(sigma_threshold) - float(np.log(n_trials))))


def width_searched(w: int, z_step: int = 1, log_sampling: bool = False) -> bool:
    """Is width w (drift z = w − 1) searched for candidates?  PAPER.md:L152, L411, Alg. 4; reading R28."""
    return bool(_load().orc_width_searched(int(w), int(z_step), int(bool(log_sampling))))


def search(spectra, zmax: int, norm_block: int, block_width: int, sigma_threshold: float, n_trials: float = 1.0,
           n_bins: int | None = None, z_step: int = 1, log_sampling: bool = False, r_block: bool = False) -> np.ndarray:
    """The whole path.  spectra: complex64 [batch, pitch] (or 1-D); n_bins defaults to the row length.
    z_step / log_sampling restrict the widths that are searched; default: every width.
    r_block: report the candidate block's first bin instead of the exact bin ("Pulscan R-Block").

    Returns a structured array (CANDIDATE_DTYPE) sorted by (spectrum, bin): at most one record per candidate block.
    """
    s = np.ascontiguousarray(spectra, dtype=np.complex64)
    if s.ndim == 1:
        s = s[None, :]
    batch, pitch = s.shape
    n = pitch if n_bins is None else int(n_bins)
    C = int(block_width)
    cap = batch * ((n + C - 1) // C)
    out = np.zeros(cap, dtype=CANDIDATE_DTYPE)
    f = s.view(np.float32)
    found = _load().orc_search_ex(f.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), batch, n, pitch, int(zmax),
                                  int(norm_block), C, float(sigma_threshold), float(n_trials), int(z_step),
                                  int(bool(log_sampling)), int(bool(r_block)), out.ctypes.data_as(ctypes.c_void_p), cap)
    return out[: int(found)].copy()


def harmonic_sum(P, H: int) -> np.ndarray:
    """Y_H(r) = sum over h = 1..H of the h adjacent powers starting at h·r (§2.3); floor(n/H) bins (R29)."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    Y = np.empty(P.size // int(H), dtype=np.float64)
    nH = _load().orc_harmonic_sum(_dp(P), P.size, int(H), _dp(Y))
    assert nH == Y.size
    return Y


def search_harmonics(spectra, zmax: int, norm_block: int, block_width: int, sigma_threshold: float, numharm: int,
                     n_trials: float = 1.0, n_bins: int | None = None, z_step: int = 1, log_sampling: bool = False,
                     r_block: bool = False, median_of_medians: bool = False, per_width: bool = False,
                     poly_logp: bool = False) -> np.ndarray:
    """The search on every harmonic-summed spectrum Y_1 … Y_numharm (§2.3): records carry `numharm`; ordered by
    (numharm, spectrum, bin); at most one per candidate block of each summed spectrum — or, with per_width, one per
    (block, searched width) above the threshold (Alg. 4), ordered by (numharm, spectrum, block, width).
    poly_logp: every ln p from Alg. 3's polynomial instead of the exact χ² tail."""
    s = np.ascontiguousarray(spectra, dtype=np.complex64)
    if s.ndim == 1:
        s = s[None, :]
    batch, pitch = s.shape
    n = pitch if n_bins is None else int(n_bins)
    C = int(block_width)
    cap = sum(batch * ((n // H + C - 1) // C) for H in range(1, int(numharm) + 1)) * (int(zmax) if per_width else 1)
    out = np.zeros(cap, dtype=CANDIDATE_DTYPE)
    f = s.view(np.float32)
    found = _load().orc_search_all(f.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), batch, n, pitch, int(zmax),
                                   int(norm_block), C, float(sigma_threshold), float(n_trials), int(z_step),
                                   int(bool(log_sampling)), int(bool(r_block)), int(numharm),
                                   int(bool(median_of_medians)), int(bool(per_width)), int(bool(poly_logp)),
                                   out.ctypes.data_as(ctypes.c_void_p), cap)
    return out[: int(found)].copy()


def median_of_medians(values) -> float:
    """Alg. 1's reduction of 4^k or 2·4^k values (reading R30); the input is not modified."""
    v = np.array(values, dtype=np.float64)
    return float(_load().orc_median_of_medians(_dp(v), v.size))


def normalise_power_mom(spectrum, norm_block: int) -> np.ndarray:
    """Steps 1-3 with the paper's GPU normalisation (Alg. 1: approximate median and MAD, scale 1.4826)."""
    f = _as_interleaved(spectrum).reshape(-1)
    n = f.size // 2
    P = np.empty(n, dtype=np.float64)
    _load().orc_normalise_power_mom(f.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), n, int(norm_block), _dp(P))
    return P

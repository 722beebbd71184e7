"""ctypes binding of libpulscan.so: the same names as include/pulscan.h, argument marshalling only.

PyTorch is used for device memory and streams; every step of the search runs in the CUDA kernels of the library.
If the library cannot be loaded this module raises — there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional

import numpy as np
import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libpulscan.so"

PULSCAN_OK, PULSCAN_EINVAL, PULSCAN_ENOWORKSPACE, PULSCAN_ECUDA, PULSCAN_EARCH = 0, -1, -2, -3, -4

CANDIDATE_DTYPE = np.dtype([("spectrum", "<i4"), ("bin", "<i4"), ("width", "<i4"), ("power", "<f4"), ("sigma", "<f4")])
assert CANDIDATE_DTYPE.itemsize == 20
HCANDIDATE_DTYPE = np.dtype([("spectrum", "<i4"), ("bin", "<i4"), ("width", "<i4"), ("numharm", "<i4"), ("power", "<f4"),
                             ("sigma", "<f4")])
assert HCANDIDATE_DTYPE.itemsize == 24

# name → (restype, argtypes); the single source for the loader and for the exported-symbol test
_P = ctypes.c_void_p
SIGNATURES = {
    "pulscan_plan_create": (_P, [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_float]),
    "pulscan_plan_set_norm_block": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_set_trials": (ctypes.c_int, [_P, ctypes.c_double]),
    "pulscan_plan_set_pitch": (ctypes.c_int, [_P, ctypes.c_int64]),
    "pulscan_plan_set_mode": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_set_width_sampling": (ctypes.c_int, [_P, ctypes.c_int32, ctypes.c_int32]),
    "pulscan_plan_set_normalisation": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_set_r_block": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_set_significance": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_set_emission": (ctypes.c_int, [_P, ctypes.c_int32, ctypes.c_int64]),
    "pulscan_plan_set_harmonics": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_max_hcandidates": (ctypes.c_int64, [_P]),
    "pulscan_search_harmonics": (ctypes.c_int, [_P, _P, _P, _P, _P]),
    "pulscan_plan_set_tuning": (ctypes.c_int, [_P, ctypes.c_int32, ctypes.c_double]),
    "pulscan_plan_set_cell_capacity": (ctypes.c_int, [_P, ctypes.c_int64]),
    "pulscan_plan_set_variant": (ctypes.c_int, [_P, ctypes.c_int32, ctypes.c_int32]),
    "pulscan_plan_max_candidates": (ctypes.c_int64, [_P]),
    "pulscan_plan_workspace_bytes": (ctypes.c_size_t, [_P]),
    "pulscan_plan_enable_host_staging": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_set_workspace": (ctypes.c_int, [_P, _P, ctypes.c_size_t]),
    "pulscan_search": (ctypes.c_int, [_P, _P, _P, _P, _P]),
    "pulscan_search_host": (ctypes.c_int, [_P, _P, _P, _P, _P]),
    "pulscan_normalise_power": (ctypes.c_int, [_P, _P, _P, _P]),
    "pulscan_plan_power_pitch": (ctypes.c_int64, [_P]),
    "pulscan_normalise_power_static": (ctypes.c_int, [_P, _P, _P, _P]),
    "pulscan_normalise_group_sums": (ctypes.c_int, [_P, _P, _P, _P, _P]),
    "pulscan_plan_group_pitch": (ctypes.c_int64, [_P]),
    "pulscan_plan_get_thresholds": (ctypes.c_int, [_P, _P]),
    "pulscan_plan_describe": (ctypes.c_int64, [_P, _P, ctypes.c_int64]),
    "pulscan_plan_get_stats": (ctypes.c_int, [_P, _P, _P]),
    "pulscan_plan_launches_per_search": (ctypes.c_int32, [_P]),
    "pulscan_plan_set_profiling": (ctypes.c_int, [_P, ctypes.c_int32]),
    "pulscan_plan_get_profile": (ctypes.c_int, [_P, ctypes.c_int32, _P]),
    "pulscan_plan_destroy": (ctypes.c_int, [_P]),
    "pulscan_last_error": (ctypes.c_char_p, []),
    "pulscan_version": (ctypes.c_char_p, []),
}

# pulscan_plan_set_variant selectors (include/pulscan.h)
VARIANT_SWEEP_SECOND_LOOK, VARIANT_SCAN_QUADS, VARIANT_NORM_KEEP_INDICES, VARIANT_NORM_L2_AHEAD = 1, 2, 3, 4
VARIANT_NORM_SINGLE_HISTOGRAM, VARIANT_KEEP_POWER = 5, 6

_lib = None


class PulscanError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"pulscan error {code}: {message}")
        self.code = code


def load_library() -> ctypes.CDLL:
    """Load libpulscan.so (built in-tree by paper_2406_15186_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(f"{LIB_PATH} not found: build it with `python -m paper_2406_15186_b200.build` "
                                    "(no CPU fallback exists)")
        lib = ctypes.CDLL(str(LIB_PATH))
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def last_error() -> str:
    return load_library().pulscan_last_error().decode()


def _check(rc: int) -> None:
    if rc != PULSCAN_OK:
        raise PulscanError(rc, last_error())


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


class Plan:
    """Owns a pulscan_plan and its torch-allocated workspace.  Thin: every method is one C-ABI call."""

    def __init__(self, n_bins: int, batch: int, zmax: int, block_width: int, sigma_threshold: float,
                 norm_block: Optional[int] = None, n_trials: Optional[float] = None, pitch: Optional[int] = None,
                 mode: int = 0, tile: int = 0, log10_p_flag: float = 0.0, host_staging: bool = False,
                 cell_capacity: int = 0, z_step: int = 1, log_sampling: bool = False, r_block: bool = False, numharm: int = 1,
                 median_of_medians: bool = False, per_width_capacity: int = 0, poly_logp: bool = False,
                 variants: Optional[dict] = None):
        self.lib = load_library()
        self.n_bins, self.batch, self.zmax, self.block_width = int(n_bins), int(batch), int(zmax), int(block_width)
        self.handle = self.lib.pulscan_plan_create(n_bins, batch, zmax, block_width, sigma_threshold)
        if not self.handle:
            raise PulscanError(PULSCAN_EINVAL, last_error())
        if norm_block is not None:
            _check(self.lib.pulscan_plan_set_norm_block(self.handle, norm_block))
        if n_trials is not None:
            _check(self.lib.pulscan_plan_set_trials(self.handle, n_trials))
        if pitch is not None:
            _check(self.lib.pulscan_plan_set_pitch(self.handle, pitch))
        if mode:
            _check(self.lib.pulscan_plan_set_mode(self.handle, mode))
        if tile or log10_p_flag:
            _check(self.lib.pulscan_plan_set_tuning(self.handle, tile, log10_p_flag))
        if host_staging:
            _check(self.lib.pulscan_plan_enable_host_staging(self.handle, 1))
        if z_step != 1 or log_sampling:
            _check(self.lib.pulscan_plan_set_width_sampling(self.handle, z_step, int(bool(log_sampling))))
        if r_block:
            _check(self.lib.pulscan_plan_set_r_block(self.handle, 1))
        if per_width_capacity:
            _check(self.lib.pulscan_plan_set_emission(self.handle, 1, per_width_capacity))
        self.capacity = int(per_width_capacity)
        if median_of_medians:
            _check(self.lib.pulscan_plan_set_normalisation(self.handle, 1))
        if poly_logp:
            _check(self.lib.pulscan_plan_set_significance(self.handle, 1))
        if numharm != 1:
            _check(self.lib.pulscan_plan_set_harmonics(self.handle, numharm))
        self.numharm = int(numharm)
        self.d_hcandidates = None
        if cell_capacity:
            _check(self.lib.pulscan_plan_set_cell_capacity(self.handle, cell_capacity))
        for which, value in (variants or {}).items():
            _check(self.lib.pulscan_plan_set_variant(self.handle, which, value))
        self.pitch = int(pitch) if pitch is not None else self.n_bins
        self.workspace = None
        self.d_candidates = None
        self.d_count = None

    # ---- host-only introspection
    @property
    def max_candidates(self) -> int:
        return int(self.lib.pulscan_plan_max_candidates(self.handle))

    @property
    def workspace_bytes(self) -> int:
        return int(self.lib.pulscan_plan_workspace_bytes(self.handle))

    @property
    def power_pitch(self) -> int:
        return int(self.lib.pulscan_plan_power_pitch(self.handle))

    @property
    def launches_per_search(self) -> int:
        return int(self.lib.pulscan_plan_launches_per_search(self.handle))

    def thresholds(self) -> np.ndarray:
        T = np.empty(self.zmax, dtype=np.float64)
        _check(self.lib.pulscan_plan_get_thresholds(self.handle, T.ctypes.data))
        return T

    def describe(self) -> str:
        need = int(self.lib.pulscan_plan_describe(self.handle, None, 0))
        if need < 0:
            raise PulscanError(PULSCAN_EINVAL, last_error())
        buf = ctypes.create_string_buffer(need)
        self.lib.pulscan_plan_describe(self.handle, ctypes.cast(buf, ctypes.c_void_p), need)
        return buf.value.decode()

    def set_mode(self, mode: int) -> None:
        """0 pruned, 1 exhaustive.  The workspace layout follows the mode (the exhaustive sweep keeps the per-bin power array),
        so an attached plan is attached again."""
        _check(self.lib.pulscan_plan_set_mode(self.handle, mode))
        if self.workspace is not None:
            self.attach(self.workspace.device)

    # ---- device side
    def attach(self, device="cuda") -> "Plan":
        """Allocate (torch) and attach the workspace and the output buffers."""
        dev = torch.device(device)
        self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=dev)
        _check(self.lib.pulscan_plan_set_workspace(self.handle, self.workspace.data_ptr(), self.workspace.numel()))
        self.d_candidates = torch.empty(self.max_candidates * CANDIDATE_DTYPE.itemsize, dtype=torch.uint8, device=dev)
        self.d_count = torch.zeros(1, dtype=torch.int32, device=dev)
        return self

    def search(self, d_spectra: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> None:
        """pulscan_search on the current (or given) stream; asynchronous.  Results stay in d_candidates / d_count."""
        if self.workspace is None:
            self.attach(d_spectra.device)
        assert d_spectra.is_cuda and d_spectra.dtype == torch.complex64 and d_spectra.is_contiguous()
        assert d_spectra.numel() >= (self.batch - 1) * self.pitch + self.n_bins
        _check(self.lib.pulscan_search(self.handle, d_spectra.data_ptr(), self.d_candidates.data_ptr(),
                                       self.d_count.data_ptr(), _stream_ptr(stream)))

    @property
    def max_hcandidates(self) -> int:
        return int(self.lib.pulscan_plan_max_hcandidates(self.handle))

    def search_harmonics(self, d_spectra: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> None:
        """pulscan_search_harmonics on the current (or given) stream; asynchronous.  Results stay in d_hcandidates / d_count."""
        if self.workspace is None:
            self.attach(d_spectra.device)
        if self.d_hcandidates is None:
            self.d_hcandidates = torch.empty(self.max_hcandidates * HCANDIDATE_DTYPE.itemsize, dtype=torch.uint8,
                                             device=d_spectra.device)
        assert d_spectra.is_cuda and d_spectra.dtype == torch.complex64 and d_spectra.is_contiguous()
        assert d_spectra.numel() >= (self.batch - 1) * self.pitch + self.n_bins
        _check(self.lib.pulscan_search_harmonics(self.handle, d_spectra.data_ptr(), self.d_hcandidates.data_ptr(),
                                                 self.d_count.data_ptr(), _stream_ptr(stream)))

    def hcandidates(self) -> np.ndarray:
        """Synchronise and return the records of the last search_harmonics, sorted by (numharm, spectrum, bin)."""
        n = self.last_count = int(self.d_count.item())
        n = min(n, self.capacity) if self.capacity else n
        raw = self.d_hcandidates[: n * HCANDIDATE_DTYPE.itemsize].cpu().numpy()
        rec = raw.view(HCANDIDATE_DTYPE).copy()
        return rec[np.lexsort((rec["width"], rec["bin"], rec["spectrum"], rec["numharm"]))]

    def candidates(self) -> np.ndarray:
        """Synchronise and return the records of the last search, sorted by (spectrum, bin)."""
        n = self.last_count = int(self.d_count.item())     # with per-width emission: the number found, possibly > capacity
        n = min(n, self.capacity) if self.capacity else n
        raw = self.d_candidates[: n * CANDIDATE_DTYPE.itemsize].cpu().numpy()
        rec = raw.view(CANDIDATE_DTYPE).copy()
        return rec[np.lexsort((rec["width"], rec["bin"], rec["spectrum"]))]

    def search_host(self, h_spectra: torch.Tensor, h_candidates: Optional[np.ndarray] = None,
                    stream: Optional[torch.cuda.Stream] = None) -> np.ndarray:
        """pulscan_search_host: host buffers in, host records out (synchronises)."""
        if self.workspace is None:
            self.attach("cuda")
        assert not h_spectra.is_cuda and h_spectra.dtype == torch.complex64 and h_spectra.is_contiguous()
        if h_candidates is None:
            h_candidates = np.empty(self.max_candidates, dtype=CANDIDATE_DTYPE)
        cnt = ctypes.c_uint32(0)
        _check(self.lib.pulscan_search_host(self.handle, h_spectra.data_ptr(), h_candidates.ctypes.data,
                                            ctypes.addressof(cnt), _stream_ptr(stream)))
        self.last_count = int(cnt.value)                     # with per-width emission: the number found, possibly > capacity
        rec = h_candidates[: min(self.last_count, self.capacity) if self.capacity else self.last_count]
        return rec[np.lexsort((rec["width"], rec["bin"], rec["spectrum"]))]

    def normalise_power(self, d_spectra: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        """Steps 1-2 only: float32 power [batch, n_bins] (a view of the padded [batch, power_pitch] buffer)."""
        out = torch.empty((self.batch, self.power_pitch), dtype=torch.float32, device=d_spectra.device)
        _check(self.lib.pulscan_normalise_power(self.handle, d_spectra.data_ptr(), out.data_ptr(), _stream_ptr(stream)))
        return out[:, : self.n_bins]

    def normalise_power_static(self, d_spectra: torch.Tensor, out: torch.Tensor,
                               stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        """pulscan_normalise_power_static: steps 1-2 for callers that cannot allocate device memory (all of it was given out
        at start-up, or the host application owns the allocator).  The plan needs no workspace and nothing is allocated here
        either: `out` is the caller's float32 [batch, power_pitch] buffer; the kernels' scratch is a fixed array inside the
        library (limit: batch x normalisation blocks <= PULSCAN_STATIC_MAX_NORM_BLOCKS).  Calls share that array: do not let
        two of them overlap on the GPU.  Returns the [batch, n_bins] view of `out`."""
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.shape == (self.batch, self.power_pitch)
        _check(self.lib.pulscan_normalise_power_static(self.handle, d_spectra.data_ptr(), out.data_ptr(), _stream_ptr(stream)))
        return out[:, : self.n_bins]

    def normalise_group_sums(self, d_spectra: torch.Tensor, norm_block: int, stream: Optional[torch.cuda.Stream] = None):
        """Steps 1-2 as the default search keeps them: (G [batch, ceil(n/4)], stats [batch, nb, 8])."""
        pitch = int(self.lib.pulscan_plan_group_pitch(self.handle))
        nb = max(1, self.n_bins // int(norm_block))
        G = torch.empty((self.batch, pitch), dtype=torch.float32, device=d_spectra.device)
        st = torch.zeros((self.batch, nb, 8), dtype=torch.float32, device=d_spectra.device)
        _check(self.lib.pulscan_normalise_group_sums(self.handle, d_spectra.data_ptr(), G.data_ptr(), st.data_ptr(),
                                                     _stream_ptr(stream)))
        return G[:, : (self.n_bins + 3) // 4], st

    def stats(self, stream: Optional[torch.cuda.Stream] = None) -> np.ndarray:
        h = np.zeros(16, dtype=np.uint32)
        _check(self.lib.pulscan_plan_get_stats(self.handle, h.ctypes.data, _stream_ptr(stream)))
        return h

    def set_profiling(self, n_slots: int) -> None:
        _check(self.lib.pulscan_plan_set_profiling(self.handle, n_slots))

    def profile(self, slot: int) -> np.ndarray:
        """Milliseconds of {memsets, kernel (a), kernel (b), kernel (c)} of the search recorded in `slot`."""
        ms = np.zeros(4, dtype=np.float32)
        _check(self.lib.pulscan_plan_get_profile(self.handle, slot, ms.ctypes.data))
        return ms

    def destroy(self) -> None:
        if getattr(self, "handle", None):
            self.lib.pulscan_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def version() -> str:
    return load_library().pulscan_version().decode()

"""Upstream stage on the same stream: dedispersed time series → cuFFT real FFT → pulscan_search, nothing leaving the GPU.

The paper's setting is a pipeline whose previous stage hands the Fourier spectrum over in device memory (PAPER.md:L39
AstroAccelerate; L346 "preallocated memory locations", L552 no transfers in the GPU timings).  Here that stage is cuFFT's
real-to-complex transform through `torch.fft.rfft` (library code: plumbing, not part of the hot path): it is enqueued on
the caller's current stream, the search is enqueued right behind it on the same stream, and the spectrum buffer is the
search's input as it stands (complex64 [batch, n_samples/2 + 1], dense rows).  No synchronisation, no host copy.
"""
from __future__ import annotations

from typing import Optional

import torch

from .binding import Plan


def search_time_series(plan: Plan, d_series: torch.Tensor, stream: Optional[torch.cuda.Stream] = None,
                       harmonics: bool = False) -> torch.Tensor:
    """Enqueue rfft + search for a batch of real float32 time series [batch, n_samples] (n_samples even,
    n_samples/2 + 1 == plan.n_bins).  Returns the spectrum tensor (kept alive by the caller until the stream has
    passed the search); results are read with plan.candidates() / plan.hcandidates()."""
    assert d_series.is_cuda and d_series.dtype == torch.float32 and d_series.dim() == 2
    assert d_series.shape[0] == plan.batch and d_series.shape[1] // 2 + 1 == plan.n_bins and d_series.shape[1] % 2 == 0
    s = stream if stream is not None else torch.cuda.current_stream()
    with torch.cuda.stream(s):
        spectrum = torch.fft.rfft(d_series, dim=1).contiguous()     # cuFFT R2C on stream s
        (plan.search_harmonics if harmonics else plan.search)(spectrum, s)
    return spectrum

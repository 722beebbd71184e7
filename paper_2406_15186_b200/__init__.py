"""pulscan-b200: the data-parallel hot path of Pulscan (arXiv 2406.15186) as hand-written sm_100a CUDA behind a C ABI.

`Plan` / `search` (in `binding`) marshal arguments into `libpulscan.so`; every step of the path runs in CUDA kernels.
`synth` holds the seeded input generators.  Importing the package does not load the CUDA library; creating a `Plan`
does, and fails loudly if it is missing — there is no CPU fallback.
"""
__version__ = "0.1.0"

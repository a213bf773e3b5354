"""paper_2606_13501_b200 — one DiT denoising step (GF-DiT's dominant computation)
as hand-written sm_100a CUDA behind a C-ABI library (include/dit.h).

`synth`   seeded synthetic inputs (no method arithmetic; shared with the tests' oracle side)
`binding` thin ctypes binding over libdit_b200.so (argument marshalling only)

Importing the package does not load the CUDA library; `binding.load()` does, and raises if it is missing.
"""
__all__ = ["synth", "binding"]

"""B200-native PRR (Predict, Reuse, Repair) decode hot path — arxiv/paper_2606_30389.

`paper_2606_30389_b200.prr` is the thin ctypes binding over the C-ABI library
(include/prr.h, csrc/); it loads `libprr.so` on first use and raises if the
library is missing — there is no CPU fallback.  `paper_2606_30389_b200.synth`
draws the seeded synthetic inputs and imports nothing else from this package.
"""
__all__ = ["prr", "synth"]

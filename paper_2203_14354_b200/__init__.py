"""B200-native photon-propagation hot path of arXiv 2203.14354.

`synth`   : seeded synthetic inputs (shared with the oracle; no method arithmetic)
`binding` : thin ctypes binding of the C-ABI library libdarwinopt.so (include/darwinopt.h)
"""
__all__ = ["synth", "binding"]

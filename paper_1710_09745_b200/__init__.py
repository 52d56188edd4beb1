"""B200-native block-CG (blockCGrQ) for the even-odd improved-staggered normal operator.

`synth`   -- seeded synthetic inputs (shared with the oracle's callers; no method arithmetic)
`binding` -- thin ctypes binding of the C-ABI library `libbkr.so` (include/bkr.h)
"""

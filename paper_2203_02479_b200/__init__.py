"""wcsim: B200-native hot path of the Wire-Cell LArTPC signal simulation, M = R (*) S + N
(arXiv 2203.02479, Eq. 1).  The work is done by hand-written sm_100a kernels behind the C-ABI
library declared in include/wcsim.h; `binding` is a thin ctypes layer with the same names."""

__all__ = ["binding", "synth", "build"]

"""B200-native brute-force incoherent dedispersion (the hot path of arxiv 2511.02328).

The product is the C-ABI library declared in include/ddsp.h (libddsp.so, built from
csrc/ by build.py); `binding` is the thin ctypes front end with the same names.  The
library is loaded on first use and the binding raises if it is missing -- there is no
CPU fallback.  `synth` holds the seeded input generators only.
"""
__all__ = ["binding", "synth", "build"]

"""gf8: B200-native GeoFP8 gradient codec (arXiv 2607.07494).  See DESIGN.md.

The C-ABI library (include/gf8.h, csrc/) is loaded lazily by `gf8` on first use so that the
input generators in `synth` can be imported without it."""
__all__ = ["gf8", "synth"]

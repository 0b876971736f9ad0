"""gsnfs-b200: B200-native (sm_100a) octree + RAHT hot path of GS-NFS's per-frame codec.

The CUDA library (libgsnfs.so, C ABI in include/gsnfs.h) is loaded lazily by `binding`;
importing this package or `synth` does not need it.  There is no CPU fallback: any call into
`binding` without the built library raises.
"""
__all__ = ["synth", "binding"]

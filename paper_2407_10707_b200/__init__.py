"""B200-native per-frame forward render of arXiv 2407.10707 (relightable, animatable Gaussian avatars).

The product is the C-ABI library `librga.so` (include/rga.h); `binding` is a thin ctypes layer with the same entry
points.  PyTorch is used for device memory and streams only.  There is no CPU fallback: importing `binding` without the
built library, or calling it without a CUDA device, raises."""
__all__ = ["binding", "build"]

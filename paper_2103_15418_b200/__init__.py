"""B200-native LPF hot path (Ruhe et al., arXiv 2103.15418): per-time-step quality control,
source detection, association, forced flux and dynamic-spectrum rings as hand-written CUDA
(sm_100a) behind the C-ABI in ``include/lpf.h``.

``synth``   seeded synthetic cube streams (NumPy only; shared with the test oracle)
``binding`` ctypes binding of the C-ABI (loads ``liblpf_b200.so``; no CPU fallback)
``build``   in-tree nvcc build
"""
__all__ = ["synth", "binding", "build"]

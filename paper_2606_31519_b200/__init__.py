"""RaBitQCache decode hot path for NVIDIA B200 (sm_100a).

The CUDA library is loaded lazily by `paper_2606_31519_b200.binding`; importing this package
(e.g. for `synth`, the input generator) does not require a GPU.  There is no CPU fallback:
every compute entry point raises if librbq_b200.so is missing.
"""
__all__ = ["synth", "binding"]

"""gsr — batched counterfactual-state Gaussian renderer for B200 (sm_100a).

The CUDA path lives in csrc/ behind the C ABI of include/gsr.h; `gsr` is the thin ctypes binding
(imported lazily so that `synth`, which needs numpy only, can be used without the extension).
"""
__all__ = ["synth"]

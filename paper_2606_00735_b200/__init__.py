"""paper_2606_00735_b200: B200-native (sm_100a) per-GPU MoE-layer hot path of ViBE.

The CUDA extension is loaded lazily by `paper_2606_00735_b200.binding`; importing the
package itself (e.g. for `inputs`) does not need a GPU.  There is no CPU fallback:
every compute entry point raises if libvibe.so is missing or no CUDA device exists.
"""
__all__ = ["inputs", "binding", "build"]

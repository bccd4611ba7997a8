"""B200-native hot path of the HAL QCD effective baryon block algorithm (arXiv:1604.07983).

`nbs` is the thin binding over the C-ABI library (include/nbs.h); `synth` draws the seeded
synthetic propagators.  Nothing here computes on the CPU: without the CUDA library the binding
raises.
"""

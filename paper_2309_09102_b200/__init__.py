"""B200-native batched Levenberg-Marquardt pose refinement (CppFlow, arxiv 2309.09102, sec. III-C).

The product is the C-ABI library declared in include/lm.h (built from csrc/ into liblm_b200.so);
`paper_2309_09102_b200.lm` is its thin ctypes binding (argument marshalling only) and
`paper_2309_09102_b200.workloads` the seeded synthetic input generators.  There is no CPU fallback:
using the binding without the built CUDA library raises.
"""
__all__ = ["lm", "workloads"]

"""paper_2306_01098_b200 -- B200-native multi-RHS HISQ Dslash and CG (arXiv:2306.01098 hot path).

The product is the C-ABI library `libhisq.so` (include/hisq.h; CUDA sources under csrc/).  This
package is the thin Python binding (`binding.Hisq`: argument marshalling only), the host-side index
maps (`layout`) and the seeded synthetic input generator (`inputs`).  There is no CPU fallback:
importing `binding` without a built library raises.
"""
__all__ = ["binding", "inputs", "layout", "build"]

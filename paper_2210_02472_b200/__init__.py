"""B200-native (sm_100a) direct-summation force path of BIFROST's HHS-FSI integrator
(arXiv:2210.02472): bifrost_acc, bifrost_grad, bifrost_dtmin, bifrost_pn1.

The product path is the CUDA library in csrc/ behind the C ABI of include/bifrost.h;
`binding` is the thin Python marshalling layer.  There is no CPU fallback: calling
any op without the built CUDA library raises.  `workloads` holds the seeded
synthetic input generators (no method arithmetic).
"""
__all__ = ["workloads"]

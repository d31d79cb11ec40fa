"""gcore-b200: the RLHF scoring hot path (fused LM-head log-probs + GRPO loss fwd/bwd) as
hand-written sm_100a CUDA behind a four-function C ABI (include/gcore.h).

``from paper_2507_22789_b200 import binding`` loads ``csrc/libgcore.so`` and raises if it is
missing: there is no CPU fallback.  ``inputs`` (seeded synthetic batches) needs no extension.
"""
__all__ = ["binding", "inputs", "build"]

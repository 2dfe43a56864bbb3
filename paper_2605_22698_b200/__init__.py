"""B200-native fused Clebsch-Gordan tensor product + scatter (the e3j hot path of arxiv 2605.22698).

The compute path lives in ``csrc/`` (CUDA, sm_100a) behind the C ABI declared in
``include/e3b200.h``; ``binding`` is argument marshalling only.  ``workloads`` holds the seeded
synthetic input generators (no method arithmetic).  Nothing here imports ``oracle/``.
"""

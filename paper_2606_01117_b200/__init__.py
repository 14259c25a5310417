"""HASTE hot path (group-shared fixed fan-in sparse output layer), B200-native.

`synth` (seeded input generators, no method arithmetic) imports without CUDA.
The binding (`paper_2606_01117_b200.haste`) loads the in-tree C-ABI library and
fails loudly when it is missing: there is no CPU fallback.
"""

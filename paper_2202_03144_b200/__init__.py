"""B200-native ptychographic projection cycle (ePIE-minibatch, DM, LSQML-style).

`synth` (seeded inputs) imports without the CUDA library; everything in `binding` needs
`csrc/libptycho_b200.so` and fails loudly without it (there is no CPU fallback).
"""
__all__ = ["synth", "binding", "sharded"]

"""paper_2007_14236_b200 — B200-native per-time-step hot path of a clock-driven spiking-network
simulator (arXiv 2007.14236): on-device connection builder, fused LIF+Poisson neuron update, spike
collection and delay-ring spike delivery, hand-written CUDA for sm_100a behind the C-ABI in
``include/ng.h``.  This package is a thin ctypes binding (argument marshalling only).

Importing the package does not load the CUDA library; ``paper_2007_14236_b200.binding`` does, and
fails loudly if ``libng.so`` is missing.  There is no CPU fallback.
"""
__all__ = ["workloads", "binding"]

"""B200-native coupled-oscillator RK4 hot path of arXiv:2410.19075.

``inputs`` and ``configs`` are pure numpy/stdlib (seeded synthetic inputs and
the five north-star workloads); ``binding`` loads the CUDA C-ABI library
``liboscnet.so`` and fails loudly if it is missing - there is no CPU fallback.
Nothing here imports the ``oracle`` package.
"""
__all__ = ["inputs", "configs", "binding", "build", "replicas"]

"""paper_2206_12205_b200 -- B200-native FDAS Fourier-domain convolution (libfdas).

``fdas``      thin ctypes binding over the C-ABI library (include/fdas.h); loaded lazily,
              fails loudly if the CUDA library has not been built.
``workloads`` seeded synthetic inputs (numpy only; none of the method's arithmetic).
"""
__all__ = ["fdas", "workloads"]

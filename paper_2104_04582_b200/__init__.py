"""paper_2104_04582_b200 -- the interpolated harmonic-mode summation of FastEMRIWaveforms (arXiv:2104.04582) as
hand-written sm_100a CUDA behind a C ABI (include/few.h).

    from paper_2104_04582_b200 import api      # ctypes binding of libfew_b200.so (needs a B200; no CPU fallback)
    from paper_2104_04582_b200 import synth    # seeded synthetic workloads (numpy only; shared with the test oracle)
    from paper_2104_04582_b200 import build    # in-tree nvcc build

Nothing is imported eagerly so that `synth` stays usable on a machine without the CUDA library.
"""
__all__ = ["api", "synth", "build"]

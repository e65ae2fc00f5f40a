"""B200-native SFT inner product (arXiv:2502.11823): C-ABI CUDA library + thin Python binding.

``paper_2502_11823_b200.api``        – ctypes binding of ``libsft_b200.so`` (include/sft.h); no CPU fallback.
``paper_2502_11823_b200.workloads``  – seeded synthetic inputs (numpy only; shared with the test oracle).
``paper_2502_11823_b200.build``      – compiles ``csrc/*.cu`` for sm_100a into the in-tree shared library.
"""
__all__ = ["api", "workloads", "build"]

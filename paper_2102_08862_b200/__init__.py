"""B200-native TPC time-frame tracker (arXiv:2102.08862): CUDA kernels behind a C-ABI + a thin binding.

``tracker`` is the binding (argument marshalling only), ``gen`` the seeded synthetic input generator,
``build`` the in-tree build, ``replicas`` the host logic of the N-GPU replica run.  There is no CPU fallback: the product path needs the CUDA library and a GPU.
"""
__all__ = ["tracker", "gen", "build", "replicas"]

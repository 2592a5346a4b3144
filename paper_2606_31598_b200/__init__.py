"""mfh -- B200-native block-procedural matrix-free Hamiltonian-vector product (phi = H psi).

The CUDA library (``lib/libmfh.so``, built from ``csrc/`` by ``build.py``) is loaded lazily by
``binding``; importing this package or ``inputs`` does not need a GPU.
"""
__all__ = ["inputs"]

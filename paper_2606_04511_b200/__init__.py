"""B200-native (sm_100a) implementation of SparDA's decode-time hot path (arxiv 2606.04511).

The product is ``libsparda.so`` (hand-written CUDA behind the C ABI in ``include/sparda.h``);
``binding`` is the thin ctypes layer with the same entry points, ``synth`` the seeded input
generators.  Importing this package does not load the library; ``binding.lib()`` does and fails
loudly if it is missing -- there is no CPU or PyTorch fallback.
"""

__all__ = ["binding", "synth", "build"]

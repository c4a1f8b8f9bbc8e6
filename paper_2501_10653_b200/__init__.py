"""B200-native tile-wise LISI / augLISI (arxiv 2501.10653, Eqs. 1-4).

* ``paper_2501_10653_b200.binding`` -- thin ctypes binding over the C-ABI CUDA library
  ``libiqa_tiles.so`` (``include/iqa_tiles.h``); argument marshalling only.  Importing it
  FAILS LOUDLY when the library has not been built: there is no CPU fallback.
* ``paper_2501_10653_b200.synth``   -- seeded synthetic sky pairs (inputs only, no method arithmetic).
* ``paper_2501_10653_b200.build``   -- nvcc build of the library for sm_100a.

The binding is loaded lazily so that ``synth`` can be used by the oracle's CPU-only tests
without touching the CUDA library.
"""
__all__ = ["binding", "synth", "build"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

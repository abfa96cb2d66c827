"""B200-native (sm_100a) multislice-ptychography hot path: batched mixed-state multislice
forward model, amplitude loss, hand-written adjoint and Adam update (PtyRAD, arxiv 2505.07814).

The compute lives in ``csrc/`` behind the C ABI declared in ``include/pty.h``; ``binding``
is the thin ctypes layer (argument marshalling only) and fails loudly if ``libpty.so`` has
not been built.  ``synth`` generates the seeded synthetic inputs and is importable without
the library.
"""
import importlib

__all__ = ["synth", "binding", "build"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

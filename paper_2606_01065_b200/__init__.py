"""leyline-b200: B200-native (sm_100a) splice of Leyline KV-cache directives (arxiv/paper_2606_01065).

The product is the C-ABI library ``libleyline.so`` (include/leyline.h); ``binding`` is its ctypes binding
(``leyline_plan``, ``leyline_splice``, ``leyline_rotate_inplace``).  ``synth`` holds the seeded synthetic inputs,
``harness`` the device-memory plumbing used by tests, bench.py and smoke().  Importing ``binding`` fails loudly
when the CUDA library cannot be built or loaded; there is no CPU fallback.
"""
__all__ = ["binding", "synth", "harness", "build"]


def __getattr__(name):
    if name in __all__:
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

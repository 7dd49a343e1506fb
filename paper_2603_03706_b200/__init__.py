"""B200-native (sm_100a) hot path of arXiv 2603.03706 tier 1: one adaptive Dormand-Prince RK45
step of the Landau-Lifshitz-Gilbert equation integrated together with N cavity-mode ODEs,
entirely on the device.  The product is ``libcavmag.so`` (C ABI in ``include/cavmag.h``);
``api`` is its thin ctypes binding.  There is no CPU fallback: touching ``api`` (or any
``cav_*`` name) without the built library raises ImportError.  ``build`` stays importable so
that the library can be compiled first.
"""


def __getattr__(name):
    if name == "build":
        import importlib
        return importlib.import_module(".build", __name__)
    import importlib
    api = importlib.import_module(".api", __name__)      # raises loudly if libcavmag.so is missing
    if name == "api":
        return api
    try:
        return getattr(api, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None

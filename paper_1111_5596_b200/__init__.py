"""paper_1111_5596_b200 -- B200-native site-parallel evaluation of QDP++-style lattice
expressions (arXiv:1111.5596).  Thin ctypes binding over ``libqdp_b200.so``
(C ABI: ``include/qdp_b200.h``).  PyTorch is used only for device memory and streams.

There is no CPU fallback: the first use of any name of the binding loads the built
library (``python -m paper_1111_5596_b200.build``) and raises ImportError if it is
missing; every call needs a CUDA device.  The binding is loaded on first attribute
access (not at package import) only so that the build module can be run before the
library exists.
"""


def __getattr__(name):
    import importlib
    binding = importlib.import_module(__name__ + ".binding")
    if name == "binding":
        return binding
    try:
        value = getattr(binding, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None
    globals()[name] = value
    return value


def __dir__():
    import importlib
    binding = importlib.import_module(__name__ + ".binding")
    return sorted(set(globals()) | set(binding.__all__))

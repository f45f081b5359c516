"""B200-native CloakLM cloaked-layout hot path: ctypes binding of the C-ABI CUDA library libcloak.so.

See include/cloak.h for the boundary and DESIGN.md for the design.  The binding (`.binding`) is loaded on
first attribute access so that `paper_2606_18400_b200.build` can run before the library exists; using any
cloak_* name without the built library raises ImportError -- there is no CPU fallback.
"""
import importlib

_binding = None


def __getattr__(name):
    global _binding
    if name.startswith("__"):
        raise AttributeError(name)
    if name in ("build", "binding"):  # submodules: `from paper_2606_18400_b200 import build` must not load the .so
        return importlib.import_module("." + name, __name__)
    if _binding is None:
        _binding = importlib.import_module(".binding", __name__)
    try:
        return getattr(_binding, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None

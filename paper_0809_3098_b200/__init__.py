"""B200-native (sm_100a) hot path of arXiv 0809.3098: the fp64 SSPRK(5,4) step of the
vorticity / stream-function lid-driven cavity.  See DESIGN.md and include/cavity.h.

Importing the package loads nothing native; `Cavity` (binding.py) loads libcavity.so on first use
and fails loudly if it is missing.  There is no CPU fallback.
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    if name in ("Cavity", "binding"):
        import importlib
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else binding.Cavity
    raise AttributeError(name)

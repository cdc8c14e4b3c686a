"""paper_2405_02410_b200 — B200-native semi-implicit pseudo-spectral SPDE stepper (cuPSS, arXiv 2405.02410).

The product is the C-ABI library built from ``csrc/`` (declared in ``include/pss.h``); this package
is the thin Python binding (argument marshalling only) plus the seeded workload generators.
"""
import importlib

from . import workloads  # noqa: F401

_BINDING_NAMES = ("System", "PssError", "lib", "F32", "F64", "DEALIAS_PAPER", "DEALIAS_TWO_THIRDS",
                  "DEALIAS_OFF", "SYMBOLS")


def __getattr__(name):
    # the binding is imported lazily so that `import paper_2405_02410_b200.workloads` works anywhere
    if name == "binding":
        return importlib.import_module(__name__ + ".binding")
    if name in _BINDING_NAMES:
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError(name)

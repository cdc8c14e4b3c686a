"""paper_2405_02410_b200 — B200-native semi-implicit pseudo-spectral SPDE stepper (cuPSS, arXiv 2405.02410).

The product is the C-ABI library built from ``csrc/`` (declared in ``include/pss.h``); this package
is the thin Python binding (argument marshalling only) plus the seeded workload generators.
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    # the binding loads libpss.so lazily so that `import paper_2405_02410_b200.workloads` works anywhere
    if name in ("System", "PssError", "binding", "lib", "F32", "F64",
                "DEALIAS_PAPER", "DEALIAS_TWO_THIRDS", "DEALIAS_OFF"):
        from . import binding as _b
        return _b if name == "binding" else getattr(_b, name)
    raise AttributeError(name)

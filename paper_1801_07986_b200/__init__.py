"""paper_1801_07986_b200 -- the limited first-order post-Newtonian N-body hot path of
arXiv:1801.07986 as hand-written sm_100a CUDA behind a C-ABI (include/pn.h).

    from paper_1801_07986_b200 import PN, inputs

`PN` (binding.py) is a thin ctypes marshalling layer over libpn.so; `inputs` holds the seeded
synthetic workloads.  Importing this package does not load the CUDA library; constructing a
`PN` does, and fails loudly if libpn.so has not been built or no CUDA device exists.
"""
from . import inputs  # noqa: F401


def __getattr__(name):
    if name in ("PN", "PNError", "load_library", "pn_version", "pn_bh_accel_noalloc"):
        from . import binding

        return getattr(binding, name)
    if name == "binding":
        import importlib

        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)

"""paper_2606_04771_b200: B200-native hot path of U(1)xSU(2)-symmetric two-site TDVP for the 1D
Fermi-Hubbard chain (arxiv/paper_2606_04771).

The product is the C-ABI library ``libfh_b200.so`` (include/fh_b200.h, sources in ``csrc/``);
``binding`` is a thin ctypes layer with the same names.  ``build`` compiles the library in-tree
with nvcc for sm_100a.  There is no CPU fallback and nothing here imports ``oracle/``.
"""
from . import build as _build_mod

build = _build_mod.build


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)

"""B200-native nodal DG Euler time step (arXiv 2006.15698 hot path) behind a C-ABI library.

`from paper_2006_15698_b200 import DG` loads the CUDA shared library built from csrc/;
importing the package (or its `inputs` module) alone loads nothing native.
"""


def __getattr__(name):
    if name in ("DG", "load_library", "DGError", "lib_path", "exported_symbols"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)

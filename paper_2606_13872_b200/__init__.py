"""B200-native Sparse Reference Attention (SRA) - the asymmetric attention of the
VideoRef DiT in arxiv/paper_2606_13872.

The product is the C-ABI library declared in include/sra.h (CUDA, sm_100a only);
`binding` is a thin ctypes marshalling layer with the same names.  Nothing here
falls back to a CPU or PyTorch implementation: if the CUDA library is missing
the binding raises.
"""
from . import inputs  # noqa: F401  (pure-python, no CUDA needed)

__all__ = ["inputs", "binding"]


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(__name__ + ".binding")
    raise AttributeError(name)

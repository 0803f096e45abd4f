"""B200-native color-gradient lattice Boltzmann step with ghost-node wetting (arxiv/paper_2605_30878).

The product is the C-ABI library ``liblbm_b200.so`` (``include/lbm.h``); ``binding`` is a thin
ctypes layer over it (argument marshalling only), ``workloads`` the seeded input generators.
The binding is imported lazily so that ``workloads`` stays importable on its own.
"""

__all__ = ["LBM", "LBMParams", "binding", "workloads"]


def __getattr__(name):
    if name in ("LBM", "LBMParams", "load_library"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)

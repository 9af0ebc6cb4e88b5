"""paper_2606_06255_b200 -- B200-native exact farthest point sampling with spherical-voxel pruning
(the hot path of RadiusFPS, arxiv/paper_2606_06255).

Sub-modules are imported lazily so that ``paper_2606_06255_b200.inputs`` (seeded input generators,
no method arithmetic) can be used without loading the CUDA library:

* ``inputs``   seeded synthetic clouds (shared with the oracle's tests)
* ``binding``  thin ctypes binding of the C-ABI in ``include/radiusfps.h`` (argument marshalling only)
* ``build``    nvcc build of ``csrc/`` into ``libradiusfps.so`` (in-tree)
"""
import importlib

__all__ = ["inputs", "binding", "build"]


def __getattr__(name):
    if name in __all__:
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

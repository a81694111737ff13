"""paper_2606_03014_b200 -- the confidence-gated aggregator stage of MOSAIC
(arxiv/paper_2606_03014, Sec. 4.2 and Alg. 1) as hand-written sm_100a CUDA behind a C ABI.

`mosaic` (the ctypes binding over csrc/libmosaic.so) is imported on first attribute access so
that `workloads` (input generators only) can be used on a box without the built library; any
call into the product path without the library raises.
"""
__all__ = ["mosaic", "workloads"]


def __getattr__(name):
    if name in ("mosaic", "workloads"):
        import importlib

        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

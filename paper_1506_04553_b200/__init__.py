"""B200-native soft-force (GPU) half of the P3T scheme, arXiv 1506.04553.

The product is the C-ABI library declared in include/p3t.h (hand-written
sm_100a CUDA under csrc/); `binding` is the thin Python front end with the same
call names.  `workloads` generates the seeded synthetic inputs.  Nothing here
falls back to the CPU: importing `binding` without the built library raises.
"""

__all__ = ["binding", "workloads"]


def __getattr__(name):
    if name in __all__:
        import importlib

        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

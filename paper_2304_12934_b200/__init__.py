"""tomoCAM hot path on B200: NUFFT Radon pair + MBIR iteration (arXiv 2304.12934).

The compute path lives in csrc/ (CUDA, C-ABI declared in include/tc.h); `binding` is
argument marshalling only and is imported lazily so that `inputs` can be used without it.
"""


def __getattr__(name):
    if name in ("binding",):
        import importlib
        return importlib.import_module(__name__ + ".binding")
    raise AttributeError(name)

"""B200-native ternary-weight linear layer (arxiv/paper_2606_08094, Section III-D, Eq. 4).

    from paper_2606_08094_b200 import binding as vla     # ctypes binding of libvlaternary.so
    from paper_2606_08094_b200 import synth               # seeded synthetic inputs (no arithmetic)

`binding` loads the CUDA library at import and raises if it is missing; there is no fallback path.
The attributes of `binding` are also reachable lazily as `paper_2606_08094_b200.<name>`.
"""
import importlib

__all__ = ["binding", "synth", "build"]


def __getattr__(name):
    if name in ("binding", "synth", "build"):
        return importlib.import_module("." + name, __name__)
    b = importlib.import_module(".binding", __name__)
    try:
        return getattr(b, name)
    except AttributeError:
        raise AttributeError("module %r has no attribute %r" % (__name__, name)) from None

"""B200-native gamma transport step loop with Geant4-style navigation (arxiv 1209.5235 hot path).

`workloads` (seeded input generators) is importable on any machine; the compute entry points
(`Geometry`, `nav_locate`, `nav_compute_step`, `transport_run`) live in `binding` and load the CUDA
C-ABI library `libgammanav.so` on first use -- there is no CPU fallback.
"""
from . import workloads  # noqa: F401

_LAZY = ("binding", "GammaNavError", "Geometry", "nav_locate", "nav_compute_step", "transport_run", "library_path")


def __getattr__(name):
    if name in _LAZY:
        import importlib
        b = importlib.import_module(".binding", __name__)
        return b if name == "binding" else getattr(b, name)
    raise AttributeError(name)

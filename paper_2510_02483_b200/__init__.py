"""paper_2510_02483_b200 -- B200-native (sm_100a) Llama decoder-layer forward+backward behind a C-ABI.

`binding` (ctypes over `liblsp.so`) is loaded lazily so that `synth` (seeded inputs, no arithmetic)
can be imported without the CUDA library.  There is no CPU fallback: using `binding` without the
built extension raises.
"""
__all__ = ["synth", "binding"]


def __getattr__(name):
    if name in ("binding", "synth"):
        import importlib
        return importlib.import_module(f"{__name__}.{name}")
    raise AttributeError(name)

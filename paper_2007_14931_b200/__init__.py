"""amp4d — B200-native evaluation of the unbinned NLL of the 4D B0 -> J/psi K pi amplitude model
(Sur et al., J Big Data 8:16, 2021; Eqs. 1-12, 14).

``binding``   thin ctypes layer over the C-ABI library ``libamp4d.so`` (include/amp.h)
``workloads`` seeded synthetic input generators for BASELINE.json's configs (no model arithmetic)

The binding is imported lazily so that the input generators can be used on a box without the
CUDA library (the oracle tests do that); any use of the binding without the built library
raises — there is no CPU fallback.
"""


def __getattr__(name):
    if name == "binding":
        import importlib
        return importlib.import_module(".binding", __name__)
    raise AttributeError(name)

"""B200-native SHO projection hot path (arXiv:1905.00480): thin Python binding over libsho.so.

``paper_1905_00480_b200.workloads`` (seeded inputs) has no dependency on the CUDA library; everything
else is loaded lazily from ``paper_1905_00480_b200.binding`` and fails loudly if libsho.so is missing.
"""
from importlib import import_module as _imp

_BINDING_NAMES = (
    "Plan", "Tables", "ShoError", "lib", "lib_path", "build_library", "nsho", "index",
    "sho_project", "sho_add", "sho_project_stored", "sho_project_host", "sho_add_host",
    "rlm_index", "umatrix", "sho_transform", "sho_dmul", "sho_apply", "sho_apply_host", "sho_project_bf", "sho_add_bf", "sho_project_bf_static", "STATIC_WORK_BYTES", "sho_add_stored", "sho_project_stored1d", "sho_add_stored1d", "Tables1D",
    "DTYPE_CODES", "DECLARED_SYMBOLS", "measure_fp64_peak", "plan_for",
)


def __getattr__(name):
    if name in _BINDING_NAMES:
        return getattr(_imp(__name__ + ".binding"), name)
    if name == "workloads":
        return _imp(__name__ + ".workloads")
    raise AttributeError(name)

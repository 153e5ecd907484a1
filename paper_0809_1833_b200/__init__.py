"""paper_0809_1833_b200 -- Matching Pursuit sparse recovery (arxiv 0809.1833) written for NVIDIA B200.

    from paper_0809_1833_b200 import mp_normalize_columns, mp_recover, mp_recover_batched

The product is the C-ABI CUDA library libmp_b200.so (include/mp_b200.h, sources in csrc/); this package
is its thin binding (binding.py) plus the seeded synthetic-input generators (synth.py, numpy only).
Importing the package does not load CUDA; the first access to a binding name does, and raises if the
library is missing and cannot be built -- there is no CPU fallback.
"""
_BINDING_NAMES = {
    "mp_normalize_columns", "mp_recover", "mp_recover_noalloc", "MP_NOALLOC_MAX_M", "mp_recover_batched", "mp_recover_host", "mp_recover_batched_host",
    "mp_workspace_bytes", "mp_probe_read", "mp_correlate_batched", "mp_encode_sparse", "mp_reconstruction_error", "mp_recover_f64", "mp_normalize_columns_f64", "mp_recover_omp", "mp_pack_signs", "mp_recover_signs", "mp_recover_many", "mp_recover_signs_many", "mp_transpose_rowmajor", "mp_set_int", "mp_get_int", "mp_last_error", "mp_launch_count",
    "mp_dictionary_create", "mp_dictionary_destroy", "mp_recover_host_h", "mp_recover_batched_host_h", "Dictionary",
    "MPError", "Recovered", "MP_OK", "MP_ERR_INVALID_ARG", "MP_ERR_CUDA", "MP_ERR_UNSUPPORTED", "MP_ERR_WORKSPACE",
}


def __getattr__(name):
    if name in _BINDING_NAMES:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)

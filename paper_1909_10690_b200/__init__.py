"""B200-native exhaustive mutual-information maps (hot path of arxiv 1909.10690, "MICUDA").

The product is the C-ABI shared library built from `csrc/` (declared in `include/mi.h`);
`binding` is a thin ctypes layer with the same names.  There is no CPU fallback: using any API
function without the built CUDA library raises.  `phantoms` is the seeded input generator
(numpy only) and can be imported without the library.
"""
_API = ("mi_create", "mi_destroy", "mi_eval_batch", "mi_eval_batch_pv", "mi_map", "mi_map_range", "mi_set_option", "mi_get_option", "mi_set_tsallis_form", "mi_set_fixed_mask", "mi_last_error",
        "mi_family_matrix", "mi_index_affine", "mi_get_bins", "mi_last_timing", "mi_release_cached_memory",
        "mi_map_gradient", "mi_map_basins", "mi_compose_matrix", "mi_seed_from_map", "mi_multimetric_gradient", "mi_register", "mi_probe_shared_atomic_rate", "mi_probe_gather_rate", "mi_version", "MIContext", "MIError")


def __getattr__(name):
    if name in _API or name == "binding":
        import importlib
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)

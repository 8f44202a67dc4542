"""B200-native ScalingAttention hot path: bit-wise block-sparse attention forward (crm kernel).

`paper_2606_23019_b200.inputs` holds the seeded input generators; everything else (the C-ABI
binding to the CUDA library) is loaded lazily so that CPU-only tools can import the package.
"""

_BINDING_NAMES = (
    "sa_pack_mask", "sa_block_sparse_attn_fwd", "sa_block_sparse_attn_fwd_ex",
    "sa_mask_words_per_row", "sa_pack_mask_workspace_bytes", "sa_fwd_workspace_bytes",
    "sa_fwd_host_scratch_bytes", "sa_block_sparse_attn_fwd_host",
    "sa_hot_path_host_scratch_bytes", "sa_hot_path_host", "sa_profile_enable", "sa_profile_collect", "sa_enumerate_active_blocks",
    "sa_set_fwd_variant", "sa_get_fwd_variant", "sa_last_launch_count",
    "sa_status_string", "sa_last_error", "load_library", "library_path", "SAError",
)


def __getattr__(name):
    if name in _BINDING_NAMES or name == "binding":
        import importlib
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)

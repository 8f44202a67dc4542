"""B200-native ScalingAttention hot path: bit-wise block-sparse attention forward (crm kernel).

`paper_2606_23019_b200.inputs` holds the seeded input generators; everything else (the C-ABI
binding to the CUDA library) is loaded lazily so that CPU-only tools can import the package.
"""

_BINDING_NAMES = (
    "sa_pack_mask", "sa_block_sparse_attn_fwd", "sa_block_sparse_attn_fwd_ex",
    "sa_mask_words_per_row", "sa_pack_mask_workspace_bytes", "sa_fwd_workspace_bytes",
    "sa_status_string", "sa_last_error", "sa_set_kernel", "sa_block_sparse_attn_fwd_host",
    "load_library", "library_path", "SAError",
)


def __getattr__(name):
    if name in _BINDING_NAMES or name == "binding":
        from . import binding
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)

"""B200-native differentiable spherical surfel rasteriser (hot path of arxiv/paper_2607_04127).

The product is the C-ABI library `liblgs.so` (include/lgs.h, csrc/*.cu, sm_100a only).
`binding` marshals torch tensors (device memory + streams only) into those calls.
Importing this package does not touch the oracle and does not load CUDA.
"""
from . import binding  # noqa: F401
from .batch import all_reduce_gradients, batch_gradients, frames_of_rank  # noqa: F401
from .binding import (  # noqa: F401
    LGS_TILE_W,
    LGS_TILE_H,
    LgsError,
    Sensor,
    Rasterizer,
    lgs_workspace_bytes,
    lgs_loss_workspace_bytes,
    lgs_render_forward,
    lgs_render_backward,
    lgs_workspace_bytes_batch,
    lgs_render_forward_batch,
    lgs_render_backward_batch,
    BatchRasterizer,
    LGS_MAX_FRAMES,
    lgs_loss_range_normal,
    lgs_loss_mapping,
    lgs_adam_step,
    lgs_scan_to_range_image,
    lgs_scan_to_range_image_static,
    LGS_SCAN_STATIC_MAX_PIXELS,
    lgs_prune_compact,
    lgs_prune_workspace_bytes,
    lgs_control_score,
    lgs_quantile,
    lgs_manage_workspace_bytes,
    lgs_split,
    lgs_cover_workspace_bytes,
    lgs_cover_prune_pass,
    lgs_compact,
    lgs_query,
    lgs_debug_tile_lists,
    lgs_debug_tile_lists_batch,
    lgs_debug_segmented_sort,
    lgs_debug_set_pdl,
    lgs_microbench,
    LGS_MB_FFMA,
    LGS_MB_MUFU_EX2,
    LGS_MB_RED_F32,
    LGS_MB_RED_F32X4,
    lgs_version,
    lgs_profile_enable,
    lgs_profile_read,
    lgs_profile_slot_name,
    library_path,
)

"""B200-native HMLFC decode + render hot path (arXiv 1902.09396).

The product is the C-ABI CUDA library libhmlfc_b200.so (include/hmlfc.h, sources in csrc/);
this package is its thin Python binding.  See DESIGN.md.
"""
from .binding import (  # noqa: F401
    EXPORTS, LIB_PATH, DECODE_AUTO, DECODE_QUEUE, DECODE_QUEUE_LAZY, DECODE_QUEUE_BLOCKREC, DECODE_THREAD, RENDER_AUTO, RENDER_PIXEL, RENDER_WARP, RENDER_WARP8, RENDER_CTA, RENDER_CTA_BIG, RENDER_CTA_SMALL, RENDER_CTA_1024, RENDER_CTA_512, RENDER_TILES, RENDER_TILES4, RENDER_TILES_W512, RENDER_TILES_W256, RENDER_TILES_W256X3, RENDER_FUSED, Footprint, Handle, HmlfcError, Info,
    hmlfc_decode, hmlfc_decode_views, hmlfc_decode_blocks, hmlfc_decode_views_host, hmlfc_decode_host, hmlfc_footprint_decode, hmlfc_footprint_render, hmlfc_free,
    hmlfc_last_oob_count, hmlfc_launch_count, hmlfc_load, hmlfc_render, hmlfc_render_noalloc, NOALLOC_MAX_TILES, hmlfc_render_lod, hmlfc_lod_levels, hmlfc_render_host, hmlfc_search,
    hmlfc_hierarchy, hmlfc_hierarchy_sizes, hmlfc_encode, hmlfc_encode_release_scratch, EncodeParams, EncodeStats,
    hmlfc_set_decode_variant, hmlfc_set_min_level, hmlfc_set_render_variant, lib,
)

// layout.cuh -- carve-up of fhgs_view_state::scratch (shared by api.cu and binsort.cu).
#pragma once
#include <stddef.h>
#include <stdint.h>

constexpr int SCAN_TILE = 1024;        // Gaussians per CTA of the scan+duplicate kernel
constexpr int SORT_TILE_K64 = 4096;    // pairs per CTA of a 64-bit-key onesweep pass
constexpr int SORT_TILE_K32 = 4096;    // pairs per CTA of a 32-bit-key onesweep pass
constexpr int SORT_MAX_PASSES = 8;
constexpr int TILE_GRID_MAX = 12288;   // (GW+1)*(GH+1) limit of the shared-memory tile-count path (48 KB)
constexpr int EMIT_TILE = 1024;        // instances per work unit of the balanced emission kernel

// ctrl words (uint32_t)
enum {
    CTRL_SCAN_TICKET = 0,     // dynamic CTA id of the scan+duplicate kernel
    CTRL_SCAN2_TICKET = 13,   // same, for the index-order offsets scan of the depth-pre-sorted mode
    CTRL_SORT_TICKET = 1,     // [1..8]  dynamic CTA ids, one per instance-sort pass
    CTRL_PRESORT_TICKET = 9,  // [9..12] dynamic CTA ids of the depth pre-sort passes
    CTRL_RENDER_QUEUE = 16,   // [16,17] work queue of fhgs_render (next item, finished CTAs; self-resetting)
    CTRL_FUSE_QUEUE = 18,     // [18,19] work queue of fhgs_fuse_features -- its own, so a render and a fuse on one view
                              //         state may overlap on two streams
    CTRL_ORDER_VALID = 20,    // 1 when tile_order holds the longest-first tile permutation of this view
    CTRL_WORDS = 64
};

struct ScratchLayout {
    size_t ctrl;          // uint32_t[CTRL_WORDS]
    size_t hist;          // uint32_t[SORT_MAX_PASSES][256]   instance-sort digit histograms
    size_t hist32;        // uint32_t[4][256]                 depth pre-sort digit histograms
    size_t zero_bytes;    // [0, zero_bytes) is cleared at the start of every fhgs_bin_sort
    size_t scan_status;   // uint64_t[2][scan_tiles]
    size_t sort_status;   // uint32_t[sort_tiles][256]
    size_t pre_keys[2];   // uint32_t[n]  depth bits (ping-pong)
    size_t pre_vals[2];   // uint32_t[n]  Gaussian index (ping-pong)
    size_t pre_incl;      // uint32_t[n]  inclusive prefix of tiles_touched in depth order
    size_t emit_starts;   // uint32_t[emit_tiles + 1]  first depth-ordered Gaussian of every EMIT_TILE instances
    size_t tile_diff;     // int32_t[(GW+1)*(GH+1)]  2-D difference array of the per-tile instance counts
    size_t tile_order;    // uint32_t[GW*GH]  tiles by descending instance count (work order of render / fuse)
    size_t tile_visited;  // uint32_t[GW*GH]  diagnostics of fhgs_render: instances of each tile's list walked before it stopped
    size_t scan_tiles, sort_tiles, pre_tiles, emit_tiles;
    size_t total;
};

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static inline ScratchLayout make_scratch_layout(int32_t n, uint64_t capacity, int32_t width = 0, int32_t height = 0) {
    ScratchLayout L;
    size_t off = 0;
    L.ctrl = off; off += align_up(CTRL_WORDS * 4, 256);
    L.hist = off; off += (size_t)SORT_MAX_PASSES * 256 * 4;
    L.hist32 = off; off += (size_t)4 * 256 * 4;
    L.zero_bytes = off;
    L.scan_tiles = ((size_t)n + SCAN_TILE - 1) / SCAN_TILE + 1;
    L.scan_status = off; off += align_up(2 * L.scan_tiles * 8, 256);
    L.sort_tiles = ((size_t)capacity + SORT_TILE_K64 - 1) / SORT_TILE_K64 + 1;
    L.pre_tiles = ((size_t)n + SORT_TILE_K32 - 1) / SORT_TILE_K32 + 1;
    const size_t st = L.sort_tiles > L.pre_tiles ? L.sort_tiles : L.pre_tiles;
    L.sort_status = off; off += st * 256 * 4;
    for (int i = 0; i < 2; ++i) { L.pre_keys[i] = off; off += align_up((size_t)n * 4, 256); }
    for (int i = 0; i < 2; ++i) { L.pre_vals[i] = off; off += align_up((size_t)n * 4, 256); }
    L.pre_incl = off; off += align_up((size_t)n * 4, 256);
    L.emit_tiles = ((size_t)capacity + EMIT_TILE - 1) / EMIT_TILE;
    L.emit_starts = off; off += align_up((L.emit_tiles + 1) * 4, 256);
    const size_t gw1 = (size_t)((width + 15) / 16 + 1), gh1 = (size_t)((height + 15) / 16 + 1);
    L.tile_diff = off; off += align_up(gw1 * gh1 * 4, 256);   // last: the regions above do not depend on width/height
    L.tile_order = off; off += align_up((gw1 - 1) * (gh1 - 1) * 4, 256);
    L.tile_visited = off; off += align_up((gw1 - 1) * (gh1 - 1) * 4, 256);
    L.total = align_up(off, 256);
    return L;
}

// lp_schedule.h -- the LP schedule engine's index math, shared by the host planner and the kernels.
//
// a1: the message [0, n) is cut into nb = ceil(n / block) blocks of `block` elements,
// the last one short (U6).  On one GPU a block is further cut into TILES of `tile` elements (the unit
// one CTA keeps on chip while it walks the chain rank 0 -> P-1); a tile never straddles a block
// boundary, so `block` stays the unit the pipeline is built from and small blocks really cost more
// (the alpha term of PAPER.md:89).  Tiles are numbered block by block and handed to the persistent CTAs in
// increasing order (lp_common.cuh, LpTileClaimer): at any moment the whole grid works on neighbouring tiles of
// the same few blocks, the analogue of "the entire network is fully utilized once the pipeline is filled".
// The pipeline kernels partition into small tiles ("granules") and move RUNS of consecutive granules of one block
// through their ring slots, so the unit of work can shrink towards the end of the list.
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define LP_HD __host__ __device__ __forceinline__
#else
#define LP_HD inline
#endif

struct lp_partition {
    uint64_t n;                // elements per rank
    uint64_t block;            // LP block b in elements (clamped to n, >= 1)
    uint64_t nb;               // number of blocks
    uint64_t tiles_per_block;  // ceil(block / tile)
    uint64_t n_tiles;          // total tiles
    uint32_t tile;             // elements per full tile
    uint32_t uniform;          // 1: every block but the last holds a whole number of full tiles (block % tile == 0, or
                               // one block): tile idx starts at idx * tile, no division needed
};

LP_HD lp_partition lp_make_partition(uint64_t n, uint64_t block, uint32_t tile) {
    lp_partition p;
    p.n = n;
    p.tile = tile;
    p.uniform = 1;
    if (n == 0) {
        p.block = block ? block : 1;
        p.nb = 0;
        p.tiles_per_block = 0;
        p.n_tiles = 0;
        return p;
    }
    if (block > n) block = n;  // "block > n => one block" (U6)
    p.block = block;
    p.nb = (n + block - 1) / block;
    p.tiles_per_block = (block + tile - 1) / tile;
    uint64_t last = n - (p.nb - 1) * block;  // length of the last block, 1..block
    p.n_tiles = (p.nb - 1) * p.tiles_per_block + (last + tile - 1) / tile;
    p.uniform = (p.nb == 1 || block % tile == 0) ? 1u : 0u;
    return p;
}

// Tile idx -> element range [off, off + len); `left` = tiles from idx to the end of its block (>= 1), so that
// idx .. idx + left - 1 are contiguous in memory and lie in one block (the last one may be short).
LP_HD void lp_tile_range_ex(const lp_partition &p, uint64_t idx, uint64_t &off, uint32_t &len, uint64_t &left,
                            uint64_t &block_end) {
    uint64_t k, j;  // block index, tile within the block
    if (((idx | p.tiles_per_block) >> 32) == 0) {  // the common case: a 32-bit division (64-bit ones are emulated on the GPU)
        const uint32_t k32 = (uint32_t)idx / (uint32_t)p.tiles_per_block;
        k = k32;
        j = (uint32_t)idx - k32 * (uint32_t)p.tiles_per_block;
    } else {
        k = idx / p.tiles_per_block;
        j = idx - k * p.tiles_per_block;
    }
    uint64_t bstart = k * p.block;
    uint64_t bend = bstart + p.block;
    if (bend > p.n) bend = p.n;
    off = bstart + j * (uint64_t)p.tile;
    uint64_t rem = bend - off;
    len = rem < p.tile ? (uint32_t)rem : p.tile;
    left = (rem + p.tile - 1) / p.tile;  // <= tiles_per_block - j (fewer in the short last block)
    block_end = bend;
}

LP_HD void lp_tile_range(const lp_partition &p, uint64_t idx, uint64_t &off, uint32_t &len) {
    if (p.uniform) {  // the common case (block a multiple of the tile): no division on the way to the first load
        off = idx * (uint64_t)p.tile;
        const uint64_t rem = p.n - off;
        len = rem < p.tile ? (uint32_t)rem : p.tile;
        return;
    }
    uint64_t left, bend;
    lp_tile_range_ex(p, idx, off, len, left, bend);
}

// ---- layer-wise messages (Alg. 1) -----------------------------------------------------
// One launch can carry a LIST of messages: slices [off[s], off[s] + len[s]) of the rank vectors, e.g. the
// layers of a network.  Every slice is its own LP message (own block partition, a1) and the tiles of the launch
// are numbered slice by slice in list order, so earlier slices finish first.  tile_start[s] is the index of
// slice s's first tile, tile_start[n_seg] the total.  The table travels as a kernel parameter (<= 4 KB).
#define LP_MAX_SEGS 96

struct lp_seg_table {
    uint64_t off[LP_MAX_SEGS];
    uint64_t len[LP_MAX_SEGS];
    uint64_t tile_start[LP_MAX_SEGS + 1];
    uint32_t n_seg;
};

// Tile idx of a segmented launch -> element range [off, off + len) in the rank vectors (+ `left`, `block_end` as in
// lp_tile_range_ex; a run of tiles never leaves its slice because a slice ends where its last block ends).
LP_HD void lp_seg_tile_range_ex(const lp_seg_table &st, uint64_t block, uint32_t tile, uint64_t idx, uint64_t &off,
                                uint32_t &len, uint64_t &left, uint64_t &block_end) {
    uint32_t lo = 0, hi = st.n_seg;  // tile_start[lo] <= idx < tile_start[hi]
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (st.tile_start[mid] <= idx) lo = mid;
        else hi = mid;
    }
    const lp_partition p = lp_make_partition(st.len[lo], block, tile);
    lp_tile_range_ex(p, idx - st.tile_start[lo], off, len, left, block_end);
    off += st.off[lo];
    block_end += st.off[lo];
}

LP_HD void lp_seg_tile_range(const lp_seg_table &st, uint64_t block, uint32_t tile, uint64_t idx, uint64_t &off,
                             uint32_t &len) {
    uint64_t left, bend;
    lp_seg_tile_range_ex(st, block, tile, idx, off, len, left, bend);
}

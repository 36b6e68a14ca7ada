// tables.h -- device-visible task / tile tables (step a5, north_star item 1: "flat task table").
// Internal to libreshard.so; the C ABI is include/reshard.h.
//
// A COPY TASK is one N-D box moved from one source buffer to k destination buffers.  The box is
// given as a contiguous run of run_bytes (the collapsed innermost dims) times nd "row" dims with
// per-side byte strides.  execute: one task per unit task, source = chosen sender's
// shard, destinations = every receiver's shard (the broadcast of PAPER.md:137, on chip).  pack: one
// task per unit task, destinations = k places in the message arena.  unpack: one task per
// (unit task, receiver), k = 1.
//
// A TILE is the unit of GPU work: n_rows consecutive rows (row-major over the row dims) times
// col_bytes of each row.  FAST tiles stay inside one span of the innermost row dim, so row r of
// the tile is at  base + r * stride[0]  on both sides with the bases precomputed by the host;
// GENERIC tiles carry the linear index of their first row and the device decodes every row.
#pragma once
#include <stdint.h>

#define RS_ROW_DIMS 7                    // RS_MAX_NDIM - 1: the last tensor dim is always in the run

struct alignas(16) RsTask {
    int64_t src_off;                     // byte offset of the box origin inside the source buffer
    int32_t src_buf;                     // index into the source pointer table
    int32_t k;                           // number of destinations
    int32_t dst_first;                   // first entry of this task in RsDst[]
    int32_t nd;                          // row dims in use (0: the box is one run)
    int64_t run_bytes;                   // contiguous bytes per row
    uint32_t ext[RS_ROW_DIMS + 1];       // ext[0] = innermost row dim ... ; unused = 1
    int64_t sstride[RS_ROW_DIMS + 1];    // byte strides, source side
    int64_t dstride[RS_ROW_DIMS + 1];    // byte strides, destination side (same for all k)
};

struct alignas(16) RsDst {
    int64_t off;                         // byte offset of the box origin inside the destination buffer
    int32_t buf;                         // index into the destination pointer table
    int32_t pad;
};

enum : uint32_t { RS_TILE_FAST = 1u };

struct alignas(16) RsTile {
    uint32_t task;
    uint32_t n_rows;
    uint32_t col_bytes;                  // bytes copied per row (<= run_bytes)
    uint32_t flags;
    // FAST: a = source offset of the tile's first byte relative to src_off, b = same for the destinations.
    // GENERIC: a = linear row index of the first row, b = byte offset inside the run.
    uint64_t a, b;
};

template <int NP>
struct RsPtrTableT {                     // kernel parameter: shard base pointers of one launch
    const char *src[NP];
    char *dst[NP];
};
typedef RsPtrTableT<128> RsPtrTable;     // RS_MAX_DEVICES per side: what the launch glue fills
#define RS_PTRS_SMALL 16                 // meshes of up to 16 devices per side get a 256-byte parameter instead of 2 KiB:
                                         // ~1 us less launch time, which is 10 % of a 1 MiB operation

struct RsOpDev {                         // one operation's tables in device memory
    const RsTask *tasks;
    const RsDst *dsts;
    const RsTile *tiles;
    uint32_t n_tiles;
};

// tables.h -- device-visible task tables (step a5, north_star item 1: "flat task table") and the
// PROCEDURAL tile decode shared by the kernels and the host.  Internal to libreshard.so; the C ABI
// is include/reshard.h.
//
// A COPY TASK is one N-D box moved from one source buffer to k destination buffers.  The box is
// given as a contiguous run of run_bytes (the collapsed innermost dims) times nd "row" dims with
// per-side byte strides.  execute: one task per unit task, source = chosen sender's
// shard, destinations = every receiver's shard (the broadcast of PAPER.md:137, on chip).  pack: one
// task per unit task, destinations = k places in the message arena.  unpack: one task per
// (unit task, receiver), k = 1.
//
// The plan is the slice list and nothing finer (App. B.2): its size is O(unit
// tasks), whatever the tensor size.  A TILE -- the unit of GPU work: n_rows consecutive rows times
// col_bytes of each row -- is never stored.  Every task carries the shape of its tile grid
// (RsTask::kind ...), every SEGMENT the index of its first tile; tile t of an operation is DECODED
// where it is needed (rs_find_seg + rs_tile_decode below; a few 32-bit divisions, done by the
// kernels 32 tiles at a time off the critical path).
//   SPLIT    runs longer than a tile: every row is cut into n_chunks column chunks of chunk_bytes
//   FAST     rows_per_tile consecutive rows inside one span of the innermost row dim, so row r of
//            the tile is at  base + r * stride[0]  on both sides
//   GENERIC  rows_per_tile consecutive LINEAR rows (innermost row dim shorter than a tile): the
//            tile carries the linear index of its first row and the kernels decode every row
// A SEGMENT is a set of n_members consecutive tasks with identical tile grids whose tiles are
// walked round-robin (tile u of member 0, tile u of member 1, ...): for slices that share
// destination rows this is DESTINATION ADDRESS order.  Everything else is a segment of one task.
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define RS_HD __host__ __device__ __forceinline__
#else
#define RS_HD inline
#endif

#define RS_ROW_DIMS 7                    // RS_MAX_NDIM - 1: the last tensor dim is always in the run

enum : uint32_t { RS_TILING_SPLIT = 0, RS_TILING_FAST = 1, RS_TILING_GENERIC = 2 };

struct alignas(16) RsTask {
    int64_t src_off;                     // byte offset of the box origin inside the source buffer
    int64_t run_bytes;                   // contiguous bytes per row
    int32_t src_buf;                     // index into the source pointer table
    int32_t k;                           // number of destinations
    int32_t dst_first;                   // first entry of this task in RsDst[]
    int32_t nd;                          // row dims in use (0: the box is one run)
    uint32_t kind;                       // RS_TILING_*
    uint32_t chunk_bytes;                // SPLIT: bytes per column chunk (multiple of 128, the last one shorter)
    uint32_t n_chunks;                   // SPLIT: chunks per row; else 1
    uint32_t rows_per_tile;              // FAST / GENERIC: rows of a full tile; SPLIT: 1
    uint32_t tiles_per_span;             // FAST: tiles per span of row dim 0 = ceil(ext[0] / rows_per_tile)
    uint32_t n_tiles;                    // tiles of this task
    uint32_t n_rows;                     // rows of the box = prod ext[i] (< 2^31)
    uint32_t tmap_ok;                    // RS_PATH_TMAP: 1 if the full tiles of this task match the tensor maps of its buffers
    uint32_t ext[RS_ROW_DIMS + 1];       // ext[0] = innermost row dim ... ; unused = 1
    int64_t sstride[RS_ROW_DIMS + 1];    // byte strides, source side
    int64_t dstride[RS_ROW_DIMS + 1];    // byte strides, destination side (same for all k)
};

struct alignas(16) RsDst {
    int64_t off;                         // byte offset of the box origin inside the destination buffer
    int32_t buf;                         // index into the destination pointer table
    int32_t pad;
};

struct alignas(16) RsSeg {
    uint32_t tile_begin;                 // index of the segment's first tile in the operation
    uint32_t first_task;
    uint32_t n_members;                  // tasks first_task .. first_task + n_members - 1, identical tile grids
    uint32_t tiles_each;                 // tiles per member
};

enum : uint32_t { RS_TILE_FAST = 1u, RS_TILE_TMAP = 2u, RS_TILE_K1 = 4u };   // K1: kernel-side only (kernels.cu RsDesc)

#define RS_TMAP_BUFS 16                  // tensor maps per side in the kernel parameter
#define RS_TMAP_ELEM 8                   // tensor-map element: UINT64 (the widest): boxes of up to 256 x 8 = 2048 bytes per row
struct RsTmapGeom {                      // one buffer seen as a 2-D byte matrix [rows][pitch]; boxes of box_rows x box_cols bytes
    int64_t pitch;
    uint32_t box_cols, box_rows;
    uint32_t valid, pad;
};

struct alignas(16) RsTile {              // a DECODED tile (never stored in a plan)
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
    const RsSeg *segs;
    uint32_t n_segs;
    uint32_t tile_base;                  // first tile of this launch (a slab of reshard_execute_host), else 0
    uint32_t n_tiles;                    // tiles of this launch
    uint32_t n_tasks, n_dsts;            // table sizes: small tables are staged in shared memory by the register kernel
    uint32_t seg_tiles;                  // > 0: every segment holds this many tiles, so tile t lies in segment t / seg_tiles (no search:
                                         // a plan of a thousand equal unit tasks would pay ten dependent table reads per tile)
    uint32_t early_trigger;              // 1: the grid covers every SM, so the next kernel of the stream may be launched at once
                                         // (programmatic dependent launch); 0: only when this kernel's CTAs run out of tiles
};

// ---- the decode -------------------------------------------------------------------------------

// the segment holding tile t: the last one whose tile_begin <= t
RS_HD uint32_t rs_find_seg(const RsSeg *segs, uint32_t n_segs, uint32_t t) {
    uint32_t lo = 0, hi = n_segs;        // invariant: segs[lo].tile_begin <= t, answer in [lo, hi)
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (segs[mid].tile_begin <= t) lo = mid; else hi = mid;
    }
    return lo;
}

// byte offsets of linear row `row` of a task's box over row dims first..nd-1 (row counted in those dims only)
RS_HD void rs_row_offsets(const RsTask &T, int first, uint32_t row, int64_t *so, int64_t *doff) {
    int64_t s = 0, d = 0;
#if defined(__CUDA_ARCH__)
#pragma unroll 1                         // off the critical path (once per tile, 32 tiles at a time): keep the code small
#endif
    for (int i = first; i < T.nd; i++) {
        const uint32_t e = T.ext[i], q = row / e, c = row - q * e;
        row = q;
        s += (int64_t)c * T.sstride[i];
        d += (int64_t)c * T.dstride[i];
    }
    *so = s; *doff = d;
}

// tile u (0 <= u < T.n_tiles) of task T
RS_HD RsTile rs_tile_decode(const RsTask &T, uint32_t task_id, uint32_t u) {
    RsTile t;
    t.task = task_id;
    int64_t so, doff;
    if (T.kind == RS_TILING_SPLIT) {
        const uint32_t row = u / T.n_chunks, cc = u - row * T.n_chunks;
        rs_row_offsets(T, 0, row, &so, &doff);
        const int64_t c0 = (int64_t)cc * T.chunk_bytes, left = T.run_bytes - c0;
        t.n_rows = 1;
        t.col_bytes = left < (int64_t)T.chunk_bytes ? (uint32_t)left : T.chunk_bytes;
        t.flags = RS_TILE_FAST;
        t.a = (uint64_t)(so + c0); t.b = (uint64_t)(doff + c0);
    } else if (T.kind == RS_TILING_FAST) {
        const uint32_t span = u / T.tiles_per_span, g = u - span * T.tiles_per_span;
        const uint32_t r0 = g * T.rows_per_tile, left = T.ext[0] - r0;
        rs_row_offsets(T, 1, span, &so, &doff);
        t.n_rows = left < T.rows_per_tile ? left : T.rows_per_tile;
        t.col_bytes = (uint32_t)T.run_bytes;
        t.flags = RS_TILE_FAST;
        t.a = (uint64_t)(so + (int64_t)r0 * T.sstride[0]); t.b = (uint64_t)(doff + (int64_t)r0 * T.dstride[0]);
    } else {
        const uint32_t r0 = u * T.rows_per_tile, left = T.n_rows - r0;
        t.n_rows = left < T.rows_per_tile ? left : T.rows_per_tile;
        t.col_bytes = (uint32_t)T.run_bytes;
        t.flags = 0;
        t.a = r0; t.b = 0;
    }
    return t;
}

// tile t of an operation: which task, which of its tiles
RS_HD void rs_tile_locate(const RsSeg *segs, uint32_t n_segs, uint32_t t, uint32_t *task, uint32_t *u, uint32_t seg_tiles = 0) {
    const RsSeg s = segs[seg_tiles ? t / seg_tiles : rs_find_seg(segs, n_segs, t)];
    const uint32_t v = t - s.tile_begin;
    if (s.n_members == 1) { *task = s.first_task; *u = v; return; }
    const uint32_t q = v / s.n_members;
    *task = s.first_task + (v - q * s.n_members);
    *u = q;
}

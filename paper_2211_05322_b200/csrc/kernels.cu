// kernels.cu -- the data path (steps a6, a7, a8): one persistent kernel launch per operation.
//
// What is computed (PAPER.md:88 task, PAPER.md:137 broadcast strategy, on chip): every copy task's
// box is read ONCE from its source buffer and written to each of its k destination buffers.
// reshard_execute / reshard_pack / reshard_unpack differ only in the task table they run.
//
// Five kernels (a TMA and a register design, each with a variant for unaligned layouts, and the tensor-map variant of
// the TMA ring), all sm_100a, no tensor cores (pure data movement, HBM-bound).  All of them: tiles decoded
// procedurally 32 at a time (tables.h), programmatic dependent launch (pdl_* below):
//   rs_copy_lsu   register path for 16-byte aligned layouts with short runs.  Every thread keeps 4
//                 independent 128-bit loads (ld.global.nc) in flight and stores each value k times.
//   rs_copy_shift / rs_copy_bulk_shift   the same two designs for layouts (or pointers) that are NOT
//                 16-byte aligned: 128-bit accesses on both sides, bytes realigned by a funnel shift.
//   rs_copy_bulk  TMA path (SASS: UBLKCP).  Every warp owns a ring of shared-memory slots: lane r
//                 issues cp.async.bulk global->shared for row r of the tile (mbarrier complete_tx),
//                 and once the tile has landed, cp.async.bulk shared->global to each of the k
//                 destinations (bulk_group).  No register staging, loads run LOOKAHEAD tiles ahead
//                 of the stores.  Needs 16-byte alignment of every address and length.  Write-heavy
//                 (multicast) launches are RATE MATCHED: every warp paces its tiles (pace_tile).
//   rs_copy_tmap  the same ring; full tiles of short rows move with cp.async.bulk.tensor.2d (SASS: UTMALDG /
//                 UTMASTG) through tensor maps encoded per call from the caller's pointers.
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <mutex>

#include "config.h"
#include "kernels.h"
#include "tables.h"

namespace rs {

// ------------------------------------------------------------------------------------------------
// shared device helpers

// Per-warp descriptor ring: everything one tile needs, resolved 32 tiles at a time (lane i resolves
// the warp's tile it+i: segment search -> task -> procedural tile decode (tables.h) -> base pointers),
// so the per-tile critical path has no dependent global load and no division -- one shared-memory
// broadcast read instead.  The plan holds no per-tile record: its size is O(unit tasks).
struct alignas(16) RsDesc {
    const char *src;                     // FAST: address of the tile's first source byte; GENERIC: box origin
    int64_t dst_rel;                     // FAST: tile.b; GENERIC: byte offset inside the run
    int64_t s0, d0;                      // row strides (FAST)
    uint64_t lin;                        // GENERIC: linear index of the first row; RS_TILE_K1 (FAST tile of a task with ONE receiver): the
                                         // address of the tile's first destination byte, so that the store side of the per-tile path
                                         // reads no table at all (a plan of a thousand unit tasks misses L1 on every tile's RsDst)
    uint32_t n_rows, col_bytes, flags, k, dst_first, task;
};
static_assert(sizeof(RsDesc) == 64, "descriptor ring slot");
#define RS_DESC_RING 64
static_assert(RS_DESC_RING * sizeof(RsDesc) == RS_BULK_DESC_BYTES, "config.h and the ring disagree");

// Programmatic dependent launch (sm_90+): every kernel lets the NEXT kernel of the stream be launched early
// (launch_dependents) and itself waits for the PREVIOUS kernel only where it first touches shard memory
// (griddepcontrol.wait; a no-op without a programmatic dependency).  What runs before the wait reads nothing but the
// plan's immutable tables and the kernel parameters: table staging, segment search, tile decode.  In a stream of
// resharding launches (or behind any kernel) launch latency and prologue overlap the predecessor's tail -- small
// operations are launch- and ramp-bound (config 3: 10.2 -> 8.1 us).  The trigger is given at entry when the grid
// covers every SM (the successor's CTAs then spread evenly: one beside each of ours); a grid that leaves SMs idle
// triggers only when its CTAs run out of tiles -- otherwise the successor's waiting CTAs pile up on the idle SMs,
// two and three to an SM, and run at half speed (measured: 96 CTAs, 3.2 instead of 6.1 TB/s).
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// the operation's tables as the kernel reads them: in global memory, or staged in shared memory (generic pointers)
struct RsTables {
    const RsTask *tasks;
    const RsDst *dsts;
    const RsSeg *segs;
};

template <int NP>
__device__ __forceinline__ void resolve_desc(const RsOpDev &op, const RsTables &tb, const RsPtrTableT<NP> &ptrs, uint32_t tile_index,
                                             RsDesc *out) {
    uint32_t task, u;
    rs_tile_locate(tb.segs, op.n_segs, op.tile_base + tile_index, &task, &u, op.seg_tiles);
    const RsTask *__restrict__ T = tb.tasks + task;
    const RsTile tile = rs_tile_decode(*T, task, u);
    RsDesc d;
    const char *base = ptrs.src[T->src_buf] + T->src_off;
    d.src = (tile.flags & RS_TILE_FAST) ? base + tile.a : base;
    d.dst_rel = (int64_t)tile.b;
    d.s0 = T->sstride[0]; d.d0 = T->dstride[0];
    d.lin = tile.a;
    d.n_rows = tile.n_rows; d.col_bytes = tile.col_bytes; d.flags = tile.flags;
    d.k = (uint32_t)T->k; d.dst_first = (uint32_t)T->dst_first; d.task = tile.task;
    if ((tile.flags & RS_TILE_FAST) && T->k == 1) {
        const RsDst D = tb.dsts[T->dst_first];
        d.lin = (uint64_t)(uintptr_t)(ptrs.dst[D.buf] + D.off + (int64_t)tile.b);
        d.flags |= RS_TILE_K1;
    }
    *out = d;
}

// GENERIC tiles: byte offsets of linear row `lin` (< 2^31) of a task's box, relative to the box origin on each side
__device__ __forceinline__ void generic_row(const RsTask *__restrict__ T, uint64_t lin, int64_t *so, int64_t *doff) {
    rs_row_offsets(*T, 0, (uint32_t)lin, so, doff);
}

// ------------------------------------------------------------------------------------------------
// register path

template <typename V> __device__ __forceinline__ V ld_stream(const char *p) {
    return *reinterpret_cast<const V *>(p);
}
template <> __device__ __forceinline__ uint4 ld_stream<uint4>(const char *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
template <typename V> __device__ __forceinline__ void st_stream(char *p, const V &v) {
    *reinterpret_cast<V *>(p) = v;
}
template <> __device__ __forceinline__ void st_stream<uint4>(char *p, const uint4 &v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1, %2, %3, %4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// GENERIC tiles (spans of the innermost row dim under 1 KiB): every vector decodes its own row (divisions), U loads in
// flight per lane as in the fast walk.
template <typename V, int U, int NP>
__device__ __forceinline__ void lsu_generic_tile(const RsTask *__restrict__ T, const RsDst *__restrict__ dsts, const RsPtrTableT<NP> &ptrs,
                                              const char *src, int64_t dst_rel, uint64_t lin, uint32_t total, uint32_t vpr, uint32_t k, int lane) {
    constexpr uint32_t VB = sizeof(V);
    for (uint32_t v0 = lane; v0 < total; v0 += 32 * U) {
        V data[U];
        int64_t doffs[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const uint32_t v = v0 + 32 * u;
            if (v < total) {
                const uint32_t r = v / vpr, c = v - r * vpr;
                int64_t so, doff;
                generic_row(T, lin + r, &so, &doff);
                doffs[u] = dst_rel + doff + (int64_t)c * VB;
                data[u] = ld_stream<V>(src + dst_rel + so + (int64_t)c * VB);
            }
        }
        for (uint32_t j = 0; j < k; j++) {
            const RsDst dd = dsts[j];
            char *dp = ptrs.dst[dd.buf] + dd.off;
#pragma unroll
            for (int u = 0; u < U; u++)
                if (v0 + 32 * u < total) st_stream<V>(dp + doffs[u], data[u]);
        }
    }
}

// Every WARP is an independent worker (no CTA-wide synchronisation anywhere).  Inside a tile the
// warp walks the (row, column) grid of V-sized vectors 32 at a time; (row, col) advance incrementally,
// so the only integer division is one per tile.  U loads are issued back to back, then U x k stores.
// GEN: the operation has GENERIC tiles.  Two instantiations, because the generic walk costs the fast one registers (64 per thread is
// the budget of 4 CTAs per SM): operations without GENERIC tiles -- nearly all -- run the kernel that does not contain it.
template <typename V, int U, int NP, bool GEN>
__global__ void __launch_bounds__(RS_LSU_THREADS, RS_LSU_CTAS_PER_SM)
rs_copy_lsu(const RsOpDev op, const __grid_constant__ RsPtrTableT<NP> ptrs) {
    constexpr uint32_t VB = sizeof(V);
    __shared__ RsDesc ring[RS_LSU_THREADS / 32][32];
    __shared__ uint4 staged[RS_LSU_TABLE_BYTES / 16];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = RS_LSU_THREADS / 32;
    RsDesc *descs = ring[warp];
    // worker = warp-major over the grid: consecutive tiles go to different CTAs, so an operation of a few hundred tiles
    // still spreads over every SM (and may give its launch_dependents trigger at entry)
    const uint32_t worker = warp * gridDim.x + blockIdx.x, n_workers = gridDim.x * W;
    const int n_my = worker < op.n_tiles ? (int)((op.n_tiles - worker + n_workers - 1) / n_workers) : 0;
    // Small tables (a few dozen unit tasks) are copied to shared memory first: one global-memory latency, after which
    // segment search, task fields and destination entries are shared-memory reads.
    if (op.early_trigger) pdl_launch_dependents();
    RsTables tb{op.tasks, op.dsts, op.segs};
    const uint32_t v_tasks = op.n_tasks * (uint32_t)(sizeof(RsTask) / 16), v_dsts = op.n_dsts, v_segs = op.n_segs;
    if ((v_tasks + v_dsts + v_segs) * 16u <= RS_LSU_TABLE_BYTES) {
        const uint4 *gt = reinterpret_cast<const uint4 *>(op.tasks), *gd = reinterpret_cast<const uint4 *>(op.dsts),
                    *gs = reinterpret_cast<const uint4 *>(op.segs);
        for (uint32_t i = threadIdx.x; i < v_tasks + v_dsts + v_segs; i += RS_LSU_THREADS)
            staged[i] = i < v_tasks ? __ldg(gt + i) : i < v_tasks + v_dsts ? __ldg(gd + (i - v_tasks)) : __ldg(gs + (i - v_tasks - v_dsts));
        __syncthreads();
        tb.tasks = reinterpret_cast<const RsTask *>(staged);
        tb.dsts = reinterpret_cast<const RsDst *>(staged + v_tasks);
        tb.segs = reinterpret_cast<const RsSeg *>(staged + v_tasks + v_dsts);
    }

    for (int it = 0; it < n_my; ++it) {
        if ((it & 31) == 0) {                                 // resolve the next 32 tiles of this warp
            __syncwarp();
            if (it + lane < n_my) resolve_desc(op, tb, ptrs, worker + (uint32_t)(it + lane) * n_workers, descs + lane);
            __syncwarp();
            if (it == 0) pdl_wait();                          // shard memory is touched from here on
        }
        const RsDesc *d = descs + (it & 31);
        const uint32_t n_rows = d->n_rows, k = d->k;
        const uint32_t vpr = d->col_bytes / VB;               // vectors per row
        const uint32_t total = n_rows * vpr;
        const RsDst *__restrict__ dsts = tb.dsts + d->dst_first;
        const bool fast = d->flags & RS_TILE_FAST;
        const char *src = d->src;
        const int64_t s0 = d->s0, d0 = d->d0, dst_rel = d->dst_rel;
        const RsTask *__restrict__ T = tb.tasks + d->task;
        if (GEN && !fast) {
            lsu_generic_tile<V, U, NP>(T, dsts, ptrs, src, dst_rel, d->lin, total, vpr, k, lane);
            continue;
        }
        const uint32_t q32 = 32u / vpr, r32 = 32u - q32 * vpr;   // how (row, col) move when v += 32
        uint32_t row = (uint32_t)lane / vpr, col = (uint32_t)lane - row * vpr;
        for (uint32_t v0 = lane; v0 < total; v0 += 32 * U) {
            V data[U];
            uint32_t r = row, c = col;
#pragma unroll
            for (int u = 0; u < U; u++) {                     // U independent loads in flight
                if (v0 + 32 * u < total) data[u] = ld_stream<V>(src + (int64_t)r * s0 + (int64_t)c * VB);
                r += q32; c += r32;
                if (c >= vpr) { c -= vpr; r++; }
            }
            for (uint32_t j = 0; j < k; j++) {                // read once, write k times
                char *dp;
                if (d->flags & RS_TILE_K1) dp = reinterpret_cast<char *>((uintptr_t)d->lin);
                else { const RsDst dd = dsts[j]; dp = ptrs.dst[dd.buf] + dd.off + dst_rel; }
                uint32_t r2 = row, c2 = col;                  // offsets are recomputed, not kept in registers
#pragma unroll
                for (int u = 0; u < U; u++) {
                    if (v0 + 32 * u < total) st_stream<V>(dp + (int64_t)r2 * d0 + (int64_t)c2 * VB, data[u]);
                    r2 += q32; c2 += r32;
                    if (c2 >= vpr) { c2 -= vpr; r2++; }
                }
            }
            row = r; col = c;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// shifted register path: any byte alignment on either side at 16-byte access width.
//
// A row of n bytes goes from s to d with s, d arbitrary.  The row is cut into SLOTS = the 16-byte
// ALIGNED windows of the destination it touches.  The value of a slot is assembled from the two
// aligned 16-byte source words that hold its bytes (byte-granular funnel shift).  A slot that lies
// fully inside the row is written with one 16-byte store; the at most two partial slots of a row
// (head, tail) are written with independent byte stores of the same assembled value.  A source word
// is loaded only if it contains at least one byte of the row, so a load never leaves the page of a
// byte the caller owns.  (row, slot) pairs are walked 32 at a time like the vectors of rs_copy_lsu.
// With k destinations the shift differs per destination, so the source is re-read per destination
// (L1/L2 hits).

__device__ __forceinline__ uint4 ld_word16(const char *p) {       // ld.global.nc, allocating in L1: the
    return __ldg(reinterpret_cast<const uint4 *>(p));              // neighbour slot re-reads this word
}

// bytes [delta, delta + 16) of the 32-byte window lo:hi (delta in 0..15)
__device__ __forceinline__ uint4 shift_window(const uint4 lo, const uint4 hi, uint32_t delta) {
    const bool w2 = delta & 8u, w1 = delta & 4u;
    const uint32_t b = (delta & 3u) * 8u;
    const uint32_t x0 = w2 ? lo.z : lo.x, x1 = w2 ? lo.w : lo.y, x2 = w2 ? hi.x : lo.z, x3 = w2 ? hi.y : lo.w,
                   x4 = w2 ? hi.z : hi.x, x5 = w2 ? hi.w : hi.y;
    const uint32_t y0 = w1 ? x1 : x0, y1 = w1 ? x2 : x1, y2 = w1 ? x3 : x2, y3 = w1 ? x4 : x3, y4 = w1 ? x5 : x4;
    return make_uint4(__funnelshift_r(y0, y1, b), __funnelshift_r(y1, y2, b), __funnelshift_r(y2, y3, b),
                      __funnelshift_r(y3, y4, b));
}

template <int U, int NP>
__global__ void __launch_bounds__(RS_LSU_THREADS, RS_LSU_CTAS_DEFAULT)
rs_copy_shift(const RsOpDev op, const __grid_constant__ RsPtrTableT<NP> ptrs) {
    __shared__ RsDesc ring[RS_LSU_THREADS / 32][32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = RS_LSU_THREADS / 32;
    RsDesc *descs = ring[warp];
    const uint32_t worker = warp * gridDim.x + blockIdx.x, n_workers = gridDim.x * W;
    const int n_my = worker < op.n_tiles ? (int)((op.n_tiles - worker + n_workers - 1) / n_workers) : 0;
    if (op.early_trigger) pdl_launch_dependents();

    for (int it = 0; it < n_my; ++it) {
        if ((it & 31) == 0) {
            __syncwarp();
            if (it + lane < n_my) resolve_desc(op, RsTables{op.tasks, op.dsts, op.segs}, ptrs, worker + (uint32_t)(it + lane) * n_workers, descs + lane);
            __syncwarp();
            if (it == 0) pdl_wait();
        }
        const RsDesc *d = descs + (it & 31);
        const uint32_t n_rows = d->n_rows, k = d->k, n = d->col_bytes;
        const RsDst *__restrict__ dsts = op.dsts + d->dst_first;
        const char *src = d->src;
        const int64_t s0 = d->s0, d0 = d->d0, dst_rel = d->dst_rel;
        if (!(d->flags & RS_TILE_FAST)) {                      // GENERIC tiles (rare): byte by byte
            const RsTask *__restrict__ T = op.tasks + d->task;
            const uint32_t total = n_rows * n;
            for (uint32_t v = lane; v < total; v += 32) {
                const uint32_t r = v / n, c = v - r * n;
                int64_t so, doff;
                generic_row(T, d->lin + r, &so, &doff);
                const char x = src[dst_rel + so + c];
                for (uint32_t j = 0; j < k; j++) {
                    const RsDst dd = dsts[j];
                    ptrs.dst[dd.buf][dd.off + dst_rel + doff + c] = x;
                }
            }
            continue;
        }
        const uint32_t SL = (n + 30u) >> 4;                     // slots per row: ceil((15 + n) / 16) at most
        const uint32_t total = n_rows * SL;
        const uint32_t q32 = 32u / SL, r32 = 32u - q32 * SL;   // how (row, slot) move when the index grows by 32
        for (uint32_t j = 0; j < k; j++) {
            const RsDst dd = dsts[j];
            char *dp = ptrs.dst[dd.buf] + dd.off + dst_rel;
            uint32_t row = (uint32_t)lane / SL, slot = (uint32_t)lane - row * SL;
            for (uint32_t v0 = lane; v0 < total; v0 += 32 * U) {
                uint4 val[U];
                uint32_t r = row, c = slot;
#pragma unroll
                for (int u = 0; u < U; u++) {                   // U independent slots in flight
                    if (v0 + 32 * u < total) {
                        const char *sr = src + (int64_t)r * s0;
                        const int32_t X = (int32_t)(c * 16u) - (int32_t)((uintptr_t)(dp + (int64_t)r * d0) & 15u);
                        const char *S = sr + X;                 // source of the slot's first byte (head slot: before the row)
                        const uint32_t delta = (uint32_t)((uintptr_t)S & 15u);
                        const char *A = S - delta;
                        // a word is loaded only if it holds a byte of the row (always true for a full slot)
                        const bool need_lo = A + 16 > sr && A < sr + n;
                        const bool need_hi = delta && A + 32 > sr && A + 16 < sr + n;
                        const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
                        const uint4 lo = need_lo ? ld_word16(A) : zero;
                        const uint4 hi = need_hi ? ld_word16(A + 16) : zero;
                        val[u] = shift_window(lo, hi, delta);
                    }
                    r += q32; c += r32;
                    if (c >= SL) { c -= SL; r++; }
                }
                uint32_t r2 = row, c2 = slot;
#pragma unroll
                for (int u = 0; u < U; u++) {
                    if (v0 + 32 * u < total) {
                        char *dr = dp + (int64_t)r2 * d0;
                        const int32_t X = (int32_t)(c2 * 16u) - (int32_t)((uintptr_t)dr & 15u);
                        if (X >= 0 && X + 16 <= (int32_t)n) {
                            *reinterpret_cast<uint4 *>(dr + X) = val[u];
                        } else {                                // head / tail (or a slot past the end): independent byte stores
                            const uint32_t w[4] = {val[u].x, val[u].y, val[u].z, val[u].w};
#pragma unroll
                            for (int i = 0; i < 16; i++)
                                if (X + i >= 0 && X + i < (int32_t)n) dr[X + i] = (char)(w[i >> 2] >> (8 * (i & 3)));
                        }
                    }
                    r2 += q32; c2 += r32;
                    if (c2 >= SL) { c2 -= SL; r2++; }
                }
                row = r; slot = c;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// TMA path

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t smem_dst, const void *gsrc, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_dst), "l"(gsrc), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *gdst, uint32_t smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 :: "l"(gdst), "r"(smem_src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read(int pending) {  // immediate operand: dispatch on the value
    switch (pending) {
        case 0: asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); break;
        case 1: asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); break;
        case 2: asm volatile("cp.async.bulk.wait_group.read 2;" ::: "memory"); break;
        case 3: asm volatile("cp.async.bulk.wait_group.read 3;" ::: "memory"); break;
        case 4: asm volatile("cp.async.bulk.wait_group.read 4;" ::: "memory"); break;
        case 5: asm volatile("cp.async.bulk.wait_group.read 5;" ::: "memory"); break;
        default: asm volatile("cp.async.bulk.wait_group.read 6;" ::: "memory"); break;
    }
}

__device__ __forceinline__ uint64_t global_ns() {             // 32 ns resolution, ~10 cycles (measured on B200)
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// RATE MATCHING.  HBM punishes an offered load above what it can drain: with every SM pushing a 1-read + k-write
// stream as fast as its store port allows (~65 GB/s per SM), 148 SMs offer ~9.6 TB/s and the achieved rate COLLAPSES to
// 5.2-5.8 TB/s, while an offered load equal to the roof (found before by trimming the grid to a magic 96 CTAs) holds
// 6.2-6.45 TB/s (profiles/r02_roof.md).  So every warp paces itself: a tile that moves b bytes of DRAM traffic
// (reads + k writes) may start `pace` x b nanoseconds after the previous one, pace = workers / target rate; the target
// is a fraction of the DRAM peak read from the device (api.cu).  A token bucket with a burst of two tiles: a warp
// that is behind schedule (HBM slower than the target, another kernel running beside) never waits.
// The target is a ceiling, not a promise: where HBM takes less than the launch offers (a hot chip -- after a burst of GEMMs the edge of the
// collapse lies 3-5 % lower --, another kernel beside, another box) the excess shows up as ring slots that are still being read when the warp
// wants them back (cp.async.bulk.wait_group.read blocks).  So the warp BACKS OFF: every time that wait takes longer than RS_PACE_BLOCK_NS its
// interval grows by 1/32, after 8 tiles without blocking it shrinks by 1/128 towards the configured target (additive-increase /
// multiplicative-decrease, per warp; all warps see the same congestion).  `mul` is that stretch factor in 1/1024.
__device__ __forceinline__ void pace_adapt(uint32_t &mul, uint32_t &calm, bool blocked) {
    if (blocked) { mul = mul + (mul >> 5); if (mul > 1536u) mul = 1536u; calm = 0; }
    else if (++calm >= 8u) { calm = 0; if (mul > 1024u) { mul -= (mul >> 7); if (mul < 1024u) mul = 1024u; } }
}

__device__ __forceinline__ void pace_tile(uint64_t &t_next, float pace, int burst, uint32_t traffic_bytes, int lane, uint32_t mul = 1024u) {
    const uint64_t interval = ((uint64_t)(pace * (float)traffic_bytes) * mul) >> 10;
    if (lane == 0) {
        uint64_t now = global_ns();
        while (now < t_next) {
            const uint64_t left = t_next - now;
            __nanosleep((unsigned)(left > 2000 ? 2000 : left));
            now = global_ns();
        }
        const uint64_t credit = (uint64_t)burst * interval;   // a warp behind schedule may catch up by this much at most
        const uint64_t floor = now - (now > credit ? credit : now);
        t_next = (t_next > floor ? t_next : floor) + interval;
    }
    __syncwarp();
}

// Tensor-map TMA (RS_PATH_TMAP): the shard of every buffer is described once per launch as a 2-D byte matrix
// [rows][pitch] with a box of box_rows x box_cols bytes (CUtensorMap, encoded on the host from the caller's pointers,
// passed as a __grid_constant__ parameter).  A full tile is then ONE cp.async.bulk.tensor.2d load (SASS UTMALDG) and
// one store per receiver (UTMASTG) instead of one bulk copy per row and receiver.  The box lands in shared memory
// densely, row after row -- the layout the per-row copies use -- so the two kinds of tile share the ring.
struct alignas(64) RsTmap { unsigned char opaque[128]; };      // CUtensorMap
struct RsTmapTable { RsTmap src[RS_TMAP_BUFS], dst[RS_TMAP_BUFS]; };

__device__ __forceinline__ void tmap_g2s(uint32_t smem_dst, const RsTmap *map, uint32_t x, uint32_t y, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(smem_dst), "l"(map), "r"(x), "r"(y), "r"(bar) : "memory");
}
__device__ __forceinline__ void tmap_s2g(const RsTmap *map, uint32_t x, uint32_t y, uint32_t smem_src) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];"
                 :: "l"(map), "r"(x), "r"(y), "r"(smem_src) : "memory");
}

template <int NP, bool TMAP>
__device__ __forceinline__ void bulk_body(const RsOpDev &op, const RsPtrTableT<NP> &ptrs, const RsTmapTable *tm, const int stages,
                                          const int lookahead, const uint32_t stage_bytes, const float pace, const int burst) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const uint32_t bars = smem_u32(smem) + warp * 64;                       // <= 8 mbarriers per warp
    RsDesc *descs = reinterpret_cast<RsDesc *>(smem + 1024) + warp * RS_DESC_RING;
    const uint32_t ring = smem_u32(smem) + 1024 + (uint32_t)W * RS_DESC_RING * sizeof(RsDesc) +
                          (uint32_t)warp * stages * stage_bytes;
    if (op.early_trigger) pdl_launch_dependents();
    if (lane == 0) {
        for (int s = 0; s < stages; s++) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const uint32_t worker = blockIdx.x * W + warp, n_workers = gridDim.x * W;
    const int n_my = worker < op.n_tiles ? (int)((op.n_tiles - worker + n_workers - 1) / n_workers) : 0;
    const int pending_ok = stages - lookahead - 1;            // store groups that may still read smem
    int ld_slot = 0, st_slot = 0;                             // it % stages, j % stages without dividing
    uint32_t st_parity = 0;
    uint64_t t_next = 0;                                      // rate matching: earliest start of this warp's next tile
    uint32_t pace_mul = 1024u, pace_calm = 0;                 // ... and its back-off (pace_adapt)
    const bool adapt = pace > 0.f && !(burst & 0x100);
    const int credit_tiles = burst & 0xff;

    for (int it = 0; it < n_my + lookahead; ++it) {
        if (it < n_my) {                                      // ---- load tile `it` into slot ld_slot
            if ((it & 31) == 0) {                             // resolve the next 32 tiles of this warp
                const int mine = it + lane;
                if (mine < n_my) {
                    RsDesc *dd = descs + (mine & (RS_DESC_RING - 1));
                    resolve_desc(op, RsTables{op.tasks, op.dsts, op.segs}, ptrs, worker + (uint32_t)mine * n_workers, dd);
                    if (TMAP) {                               // a full tile of a task whose buffers have tensor maps
                        const RsTask *__restrict__ T = op.tasks + dd->task;
                        if (T->tmap_ok && dd->n_rows == T->rows_per_tile) {
                            const uint64_t addr = (uint64_t)(dd->src - ptrs.src[T->src_buf]);   // byte offset inside the source buffer
                            const uint64_t y = addr / (uint64_t)dd->s0;
                            dd->lin = (y << 32) | (uint64_t)((addr - y * (uint64_t)dd->s0) / RS_TMAP_ELEM);
                            dd->task = (uint32_t)T->src_buf;
                            dd->flags = (dd->flags | RS_TILE_TMAP) & ~RS_TILE_K1;
                        }
                    }
                }
                __syncwarp();
                if (it == 0) pdl_wait();                      // shard memory is touched from here on
            }
            if (it >= stages) {                               // slot reuse: its stores must have read it
                if (adapt) {
                    const uint64_t t0 = global_ns();
                    bulk_wait_read(pending_ok);
                    pace_adapt(pace_mul, pace_calm, global_ns() - t0 > RS_PACE_BLOCK_NS);
                } else {
                    bulk_wait_read(pending_ok);
                }
                __syncwarp();
            }
            const RsDesc *d = descs + (it & (RS_DESC_RING - 1));
            const uint32_t n_rows = d->n_rows, col_bytes = d->col_bytes;
            if (pace > 0.f) pace_tile(t_next, pace, credit_tiles, n_rows * col_bytes * (1u + d->k), lane, pace_mul);
            const uint32_t bar = bars + 8 * ld_slot, slot = ring + (uint32_t)ld_slot * stage_bytes;
            if (lane == 0) mbar_expect_tx(bar, n_rows * col_bytes);
            __syncwarp();
            if (TMAP && (d->flags & RS_TILE_TMAP)) {
                if (lane == 0) tmap_g2s(slot, tm->src + d->task, (uint32_t)d->lin, (uint32_t)(d->lin >> 32), bar);
            } else if (d->flags & RS_TILE_FAST) {
                const char *src = d->src;
                const int64_t s0 = d->s0;
                if (s0 == (int64_t)col_bytes || n_rows == 1) { // rows adjacent in the source: the tile is ONE run there
                    if (lane == 0) bulk_g2s(slot, src, n_rows * col_bytes, bar);
                } else {
                    for (uint32_t r = lane; r < n_rows; r += 32)
                        bulk_g2s(slot + r * col_bytes, src + (int64_t)r * s0, col_bytes, bar);
                }
            } else {
                const RsTask *__restrict__ T = op.tasks + d->task;
                for (uint32_t r = lane; r < n_rows; r += 32) {
                    int64_t so, doff;
                    generic_row(T, d->lin + r, &so, &doff);
                    bulk_g2s(slot + r * col_bytes, d->src + d->dst_rel + so, col_bytes, bar);
                }
            }
            if (++ld_slot == stages) ld_slot = 0;
        }
        const int j = it - lookahead;
        if (j >= 0) {                                         // ---- store tile j to its k destinations
            const RsDesc *d = descs + (j & (RS_DESC_RING - 1));
            const uint32_t n_rows = d->n_rows, col_bytes = d->col_bytes, k = d->k;
            const RsDst *__restrict__ dsts = op.dsts + d->dst_first;
            const uint32_t slot = ring + (uint32_t)st_slot * stage_bytes;
            const bool fast = d->flags & RS_TILE_FAST;
            mbar_wait(bars + 8 * st_slot, st_parity);
            if (TMAP && (d->flags & RS_TILE_TMAP)) {          // lane q stores the whole box to receiver q
                for (uint32_t q = lane; q < k; q += 32) {
                    const RsDst dd = dsts[q];
                    const uint64_t addr = (uint64_t)(dd.off + d->dst_rel), y = addr / (uint64_t)d->d0;
                    tmap_s2g(tm->dst + dd.buf, (uint32_t)((addr - y * (uint64_t)d->d0) / RS_TMAP_ELEM), (uint32_t)y, slot);
                }
            } else if (fast && (d->d0 == (int64_t)col_bytes || n_rows == 1)) {
                // rows adjacent in the destinations (a message, or a shard whose rows the slice covers whole): lane q
                // stores the tile to receiver q with ONE bulk copy
                if (d->flags & RS_TILE_K1) {
                    if (lane == 0) bulk_s2g(reinterpret_cast<char *>((uintptr_t)d->lin), slot, n_rows * col_bytes);
                } else
                for (uint32_t q = lane; q < k; q += 32) {
                    const RsDst dd = dsts[q];
                    bulk_s2g(ptrs.dst[dd.buf] + dd.off + d->dst_rel, slot, n_rows * col_bytes);
                }
            } else {                                          // (rows apart: the table read stays -- taking it out made the row stores of
                                                              // P1 / P4 issue faster and the launch 3-6 % SLOWER, the open-loop effect again)
                const RsTask *__restrict__ T = op.tasks + d->task;
                for (uint32_t r = lane; r < n_rows; r += 32) {
                    int64_t doff;
                    if (fast) {
                        doff = d->dst_rel + (int64_t)r * d->d0;
                    } else {
                        int64_t so;
                        generic_row(T, d->lin + r, &so, &doff);
                        doff += d->dst_rel;
                    }
                    for (uint32_t q = 0; q < k; q++) {        // read once, write k times
                        const RsDst dd = dsts[q];
                        bulk_s2g(ptrs.dst[dd.buf] + dd.off + doff, slot + r * col_bytes, col_bytes);
                    }
                }
            }
            bulk_commit();
            if (++st_slot == stages) { st_slot = 0; st_parity ^= 1u; }
        }
    }
    pdl_launch_dependents();                                  // out of tiles: the successor may start beside the drain
    bulk_wait_read(0);                                        // shared memory must outlive the stores' reads
}

template <int NP>
__global__ void __launch_bounds__(256, 1)
rs_copy_bulk(const RsOpDev op, const __grid_constant__ RsPtrTableT<NP> ptrs, const int stages, const int lookahead,
             const uint32_t stage_bytes, const float pace, const int burst) {
    bulk_body<NP, false>(op, ptrs, nullptr, stages, lookahead, stage_bytes, pace, burst);
}

__global__ void __launch_bounds__(256, 1)
rs_copy_tmap(const RsOpDev op, const __grid_constant__ RsPtrTableT<RS_PTRS_SMALL> ptrs, const __grid_constant__ RsTmapTable tm,
             const int stages, const int lookahead, const uint32_t stage_bytes, const float pace, const int burst) {
    bulk_body<RS_PTRS_SMALL, true>(op, ptrs, &tm, stages, lookahead, stage_bytes, pace, burst);
}

// ------------------------------------------------------------------------------------------------
// TMA loads + shifted register stores: the deep asynchronous load pipeline of rs_copy_bulk for rows
// whose addresses or lengths are NOT multiples of 16 bytes.
//
// Loads: lane r asks the copy engine for the 16-byte ALIGNED superset of row r (from floor16(src) to
// ceil16(src + n): at most 15 bytes before and after the row, always inside aligned words that hold
// bytes of the row).  Row r lands at  slot + r * pitch + 16  with its first byte at (src & 15).
// Stores: once the tile has landed the warp walks the 16-byte aligned windows of every DESTINATION
// row, assembles each from two aligned shared-memory words (shift_window) and stores it with one
// st.global.v4 (head / tail windows: byte stores).  Shared-memory latency is short, so a few warps
// keep up; DRAM latency is hidden by the loads running LOOKAHEAD tiles ahead.

__device__ __forceinline__ uint32_t shift_pitch(uint32_t n) { return (n + 77u) & ~15u; }   // 16 slack + 15 + n + 46

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}

// One destination row: n bytes sit in shared memory from byte address `sm`; write them to `dr`.
// The row is cut at the destination's 16-byte boundaries: head bytes, `full` aligned windows, tail
// bytes.  The byte shift between source and destination is the same for every window of the row, so
// it is resolved ONCE per row (switch on its word part, funnel shift by its byte part): a window
// costs two ld.shared.v4, four SHF.R and one st.global.v4.
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
    uint32_t r;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}

template <int W>
__device__ __forceinline__ void row_windows(char *dst16, uint32_t base, uint32_t full, uint32_t b, uint32_t lane) {
#pragma unroll 2
    for (uint32_t c = lane; c < full; c += 32) {
        const uint4 lo = lds128(base + 16u * c), hi = lds128(base + 16u * c + 16u);
        const uint32_t w[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
        *reinterpret_cast<uint4 *>(dst16 + 16u * c) =
            make_uint4(__funnelshift_r(w[W], w[W + 1], b), __funnelshift_r(w[W + 1], w[W + 2], b),
                       __funnelshift_r(w[W + 2], w[W + 3], b), __funnelshift_r(w[W + 3], w[W + 4], b));
    }
}

__device__ __forceinline__ void store_row(char *dr, uint32_t sm, uint32_t n, uint32_t lane) {
    uint32_t head = (16u - (uint32_t)((uintptr_t)dr & 15u)) & 15u;
    if (head > n) head = n;
    const uint32_t full = (n - head) >> 4, tail = n - head - (full << 4);
    const uint32_t q0 = sm + head, delta = q0 & 15u, b = (delta & 3u) * 8u, base = q0 - delta;
    switch (delta >> 2) {                                     // warp-uniform
        case 0: row_windows<0>(dr + head, base, full, b, lane); break;
        case 1: row_windows<1>(dr + head, base, full, b, lane); break;
        case 2: row_windows<2>(dr + head, base, full, b, lane); break;
        default: row_windows<3>(dr + head, base, full, b, lane); break;
    }
    if (lane < head) dr[lane] = (char)lds_u8(sm + lane);
    else if (lane >= 16u && lane - 16u < tail) {
        const uint32_t off = head + (full << 4) + lane - 16u;
        dr[off] = (char)lds_u8(sm + off);
    }
}

// TMA STORES for unaligned rows.  cp.async.bulk needs 16-byte aligned addresses and sizes on both sides, and the
// 16-byte aligned BODY of a destination row (everything but < 16 head and < 16 tail bytes) has them in global memory.
// So the body is first realigned INSIDE the ring slot: window c of the body (row bytes [head + 16c, head + 16c + 16),
// which sit at q0 + 16c with q0 = base + delta) is assembled from the aligned words c and c + 1 and written back over
// word c.  32 windows at a time, all loads before all stores: a group overwrites words c0 .. c0 + 31 and has read words
// c0 .. c0 + 32; the next group starts at word c0 + 32, which is still intact.  Afterwards one bulk copy per row and
// receiver stores the body from `base` (st.global from registers tops out ~6 % below TMA stores on B200: DESIGN.md S3).
__device__ __forceinline__ void sts128(uint32_t addr, const uint4 &v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" :: "r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

template <int W>
__device__ __forceinline__ uint4 funnel_window(const uint4 &lo, const uint4 &hi, uint32_t b) {
    const uint32_t w[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
    return make_uint4(__funnelshift_r(w[W], w[W + 1], b), __funnelshift_r(w[W + 1], w[W + 2], b),
                      __funnelshift_r(w[W + 2], w[W + 3], b), __funnelshift_r(w[W + 3], w[W + 4], b));
}

// (one warp per scheduler hides no latency: what counts is the instruction count, so 128 windows per trip, four per lane)
template <int W>
__device__ __forceinline__ void row_realign(uint32_t base, uint32_t full, uint32_t b, uint32_t lane) {
    uint32_t c0 = 0;
    for (; c0 + 128u <= full; c0 += 128u) {                                 // whole trips: no predicates
        const uint32_t p = base + 16u * (c0 + lane);
        const uint4 l0 = lds128(p), h0 = lds128(p + 16u), l1 = lds128(p + 512u), h1 = lds128(p + 528u),
                    l2 = lds128(p + 1024u), h2 = lds128(p + 1040u), l3 = lds128(p + 1536u), h3 = lds128(p + 1552u);
        __syncwarp();
        sts128(p, funnel_window<W>(l0, h0, b));
        sts128(p + 512u, funnel_window<W>(l1, h1, b));
        sts128(p + 1024u, funnel_window<W>(l2, h2, b));
        sts128(p + 1536u, funnel_window<W>(l3, h3, b));
        __syncwarp();
    }
    for (; c0 < full; c0 += 32u) {                                          // the ragged rest, 32 windows per trip
        const uint32_t c = c0 + lane, p = base + 16u * c;
        uint4 lo, hi;
        if (c < full) { lo = lds128(p); hi = lds128(p + 16u); }
        __syncwarp();
        if (c < full) sts128(p, funnel_window<W>(lo, hi, b));
        __syncwarp();
    }
}

// where the pieces of one destination row are: n bytes in shared memory from `sm`, going to global address `dr`
struct RowCut { uint32_t head, full, tail, base, delta; };
__device__ __forceinline__ RowCut cut_row(uintptr_t dr, uint32_t sm, uint32_t n) {
    RowCut c;
    c.head = (16u - (uint32_t)(dr & 15u)) & 15u;
    if (c.head > n) c.head = n;
    c.full = (n - c.head) >> 4;
    c.tail = n - c.head - (c.full << 4);
    const uint32_t q0 = sm + c.head;
    c.delta = q0 & 15u;
    c.base = q0 - c.delta;
    return c;
}

// One 16-byte aligned window of a destination row, in two steps so that several windows' shared-memory
// loads can be in flight: n bytes of the row sit in shared memory from byte address `sm`.
struct ShiftSlot { uint4 lo, hi; int32_t X; uint32_t delta; };

__device__ __forceinline__ void slot_load(ShiftSlot &t, const char *dr, uint32_t sm, uint32_t n, uint32_t c) {
    t.X = (int32_t)(c * 16u) - (int32_t)((uintptr_t)dr & 15u);              // row byte the window starts at (>= -15)
    if (t.X >= (int32_t)n) return;                                          // window past the end of the row
    const uint32_t q = sm + (uint32_t)t.X;                                  // 16 bytes of slack precede the row
    t.delta = q & 15u;
    t.lo = lds128(q - t.delta);
    t.hi = lds128(q - t.delta + 16u);
}

__device__ __forceinline__ void slot_store(const ShiftSlot &t, char *dr, uint32_t n) {
    if (t.X >= (int32_t)n) return;
    const uint4 v = shift_window(t.lo, t.hi, t.delta);
    if (t.X >= 0 && t.X + 16 <= (int32_t)n) {
        *reinterpret_cast<uint4 *>(dr + t.X) = v;
    } else {                                                                // head / tail: independent byte stores
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 16; i++)
            if (t.X + i >= 0 && t.X + i < (int32_t)n) dr[t.X + i] = (char)(w[i >> 2] >> (8 * (i & 3)));
    }
}

template <int NP>
__global__ void __launch_bounds__(256, 1)
rs_copy_bulk_shift(const RsOpDev op, const __grid_constant__ RsPtrTableT<NP> ptrs, const int stages, const int lookahead,
                   const uint32_t stage_bytes, const int mode, const float pace, const int burst) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const uint32_t bars = smem_u32(smem) + warp * 64;
    RsDesc *descs = reinterpret_cast<RsDesc *>(smem + 1024) + warp * RS_DESC_RING;
    const uint32_t ring = smem_u32(smem) + 1024 + (uint32_t)W * RS_DESC_RING * sizeof(RsDesc) +
                          (uint32_t)warp * stages * stage_bytes;
    if (op.early_trigger) pdl_launch_dependents();
    if (lane == 0) {
        for (int s = 0; s < stages; s++) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const uint32_t worker = blockIdx.x * W + warp, n_workers = gridDim.x * W;
    const int n_my = worker < op.n_tiles ? (int)((op.n_tiles - worker + n_workers - 1) / n_workers) : 0;
    const int pending_ok = stages - lookahead - 1;            // store groups that may still read the ring (>= 0)
    int ld_slot = 0, st_slot = 0;
    uint32_t st_parity = 0;
    uint64_t t_next = 0;                                      // rate matching (pace_tile), as in rs_copy_bulk

    for (int it = 0; it < n_my + lookahead; ++it) {
        if (it < n_my) {                                      // ---- load tile `it`
            if ((it & 31) == 0) {
                const int mine = it + lane;
                if (mine < n_my)
                    resolve_desc(op, RsTables{op.tasks, op.dsts, op.segs}, ptrs, worker + (uint32_t)mine * n_workers, descs + (mine & (RS_DESC_RING - 1)));
                __syncwarp();
                if (it == 0) pdl_wait();                      // shard memory is touched from here on
            }
            if (it >= stages) {                               // slot reuse: the bulk stores of its last tile must have read it
                bulk_wait_read(pending_ok);                   // (register stores drained it in program order)
                __syncwarp();
            }
            const RsDesc *d = descs + (it & (RS_DESC_RING - 1));
            const uint32_t n_rows = d->n_rows, n = d->col_bytes, pitch = shift_pitch(n);
            if (pace > 0.f) pace_tile(t_next, pace, burst & 0xff, n_rows * n * (1u + d->k), lane);
            const uint32_t bar = bars + 8 * ld_slot, slot = ring + (uint32_t)ld_slot * stage_bytes;
            const bool fast = d->flags & RS_TILE_FAST;
            const RsTask *__restrict__ T = op.tasks + d->task;
            uint32_t my_bytes = 0;
            for (uint32_t r = lane; r < n_rows; r += 32) {     // bytes this lane will ask for
                int64_t so = (int64_t)r * d->s0, doff;
                if (!fast) { generic_row(T, d->lin + r, &so, &doff); so += d->dst_rel; }
                const uint32_t a = (uint32_t)((uintptr_t)(d->src + so) & 15u);
                my_bytes += (a + n + 15u) & ~15u;
            }
            const uint32_t tile_bytes = __reduce_add_sync(0xffffffffu, my_bytes);
            if (lane == 0) mbar_expect_tx(bar, tile_bytes);
            __syncwarp();
            for (uint32_t r = lane; r < n_rows; r += 32) {
                int64_t so = (int64_t)r * d->s0, doff;
                if (!fast) { generic_row(T, d->lin + r, &so, &doff); so += d->dst_rel; }
                const char *g = d->src + so;
                const uint32_t a = (uint32_t)((uintptr_t)g & 15u);
                bulk_g2s(slot + r * pitch + 16u, g - a, (a + n + 15u) & ~15u, bar);
            }
            if (++ld_slot == stages) ld_slot = 0;
        }
        const int j = it - lookahead;
        if (j >= 0) {                                         // ---- store tile j to its k destinations
            const RsDesc *d = descs + (j & (RS_DESC_RING - 1));
            const uint32_t n_rows = d->n_rows, n = d->col_bytes, k = d->k, pitch = shift_pitch(n);
            const RsDst *__restrict__ dsts = op.dsts + d->dst_first;
            const uint32_t slot = ring + (uint32_t)st_slot * stage_bytes;
            const bool fast = d->flags & RS_TILE_FAST;
            const RsTask *__restrict__ T = op.tasks + d->task;
            const uint32_t SL = (n + 30u) >> 4;               // destination windows per row, at most
            mbar_wait(bars + 8 * st_slot, st_parity);
            // Long rows whose k destinations are congruent modulo 16 (always, for k = 1): realign the body of every row in
            // place, then one bulk store per row and receiver; head and tail bytes go out as byte stores.
            bool tma_stores = mode == RS_SHIFT_BULK && fast && SL >= 64u && n_rows <= 32u;
            if (tma_stores && k > 1) {
                const uint32_t a0 = (uint32_t)((uintptr_t)(ptrs.dst[dsts[0].buf] + dsts[0].off) & 15u);
                bool same = true;
                for (uint32_t q = lane; q < k; q += 32) same = same && ((uint32_t)((uintptr_t)(ptrs.dst[dsts[q].buf] + dsts[q].off) & 15u) == a0);
                tma_stores = __all_sync(0xffffffffu, same);
            }
            if (tma_stores) {
                const RsDst d0q = dsts[0];
                const uintptr_t dp0 = (uintptr_t)(ptrs.dst[d0q.buf] + d0q.off + d->dst_rel);
                for (uint32_t r = 0; r < n_rows; r++) {
                    const uint32_t sm = slot + r * pitch + 16u + (uint32_t)((uintptr_t)(d->src + (int64_t)r * d->s0) & 15u);
                    const RowCut c = cut_row(dp0 + (uintptr_t)((int64_t)r * d->d0), sm, n);
                    uint32_t edge = 0;                        // this lane's head or tail byte, read before the body moves
                    const bool is_head = (uint32_t)lane < c.head, is_tail = lane >= 16 && (uint32_t)lane - 16u < c.tail;
                    const uint32_t edge_off = is_head ? (uint32_t)lane : c.head + (c.full << 4) + (uint32_t)lane - 16u;
                    if (is_head || is_tail) edge = lds_u8(sm + edge_off);
                    __syncwarp();
                    if (c.delta) {
                        const uint32_t b = (c.delta & 3u) * 8u;
                        switch (c.delta >> 2) {               // warp-uniform
                            case 0: row_realign<0>(c.base, c.full, b, (uint32_t)lane); break;
                            case 1: row_realign<1>(c.base, c.full, b, (uint32_t)lane); break;
                            case 2: row_realign<2>(c.base, c.full, b, (uint32_t)lane); break;
                            default: row_realign<3>(c.base, c.full, b, (uint32_t)lane); break;
                        }
                    }
                    if (is_head || is_tail)
                        for (uint32_t q = 0; q < k; q++) {
                            const RsDst dd = dsts[q];
                            (ptrs.dst[dd.buf] + dd.off + d->dst_rel + (int64_t)r * d->d0)[edge_off] = (char)edge;
                        }
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the realigned bodies, before the copy engine reads them
                __syncwarp();
                if ((uint32_t)lane < n_rows) {                // lane r: the body of row r to every receiver
                    const uint32_t r = (uint32_t)lane;
                    const uint32_t sm = slot + r * pitch + 16u + (uint32_t)((uintptr_t)(d->src + (int64_t)r * d->s0) & 15u);
                    const RowCut c = cut_row(dp0 + (uintptr_t)((int64_t)r * d->d0), sm, n);
                    if (c.full)
                        for (uint32_t q = 0; q < k; q++) {
                            const RsDst dd = dsts[q];
                            bulk_s2g(ptrs.dst[dd.buf] + dd.off + d->dst_rel + (int64_t)r * d->d0 + c.head, c.base, c.full << 4);
                        }
                }
            } else
            for (uint32_t q = 0; q < k; q++) {                // read once (from HBM), write k times
                const RsDst dd = dsts[q];
                char *dp = ptrs.dst[dd.buf] + dd.off + d->dst_rel;
                if (fast && SL < 64u) {                       // short rows: flat walk over (row, window), 2 in flight per lane
                    const uint32_t total = n_rows * SL, q32 = 32u / SL, r32 = 32u - q32 * SL;
                    uint32_t r = (uint32_t)lane / SL, c = (uint32_t)lane - r * SL;
                    for (uint32_t v = lane; v < total; v += 64) {
                        ShiftSlot t0, t1;
                        char *dr0 = dp + (int64_t)r * d->d0, *dr1 = dr0;
                        slot_load(t0, dr0, slot + r * pitch + 16u + (uint32_t)((uintptr_t)(d->src + (int64_t)r * d->s0) & 15u), n, c);
                        r += q32; c += r32;
                        if (c >= SL) { c -= SL; r++; }
                        const bool two = v + 32 < total;
                        if (two) {
                            dr1 = dp + (int64_t)r * d->d0;
                            slot_load(t1, dr1, slot + r * pitch + 16u + (uint32_t)((uintptr_t)(d->src + (int64_t)r * d->s0) & 15u), n, c);
                        }
                        r += q32; c += r32;
                        if (c >= SL) { c -= SL; r++; }
                        slot_store(t0, dr0, n);
                        if (two) slot_store(t1, dr1, n);
                    }
                } else {                                      // long rows: row by row, the shift is uniform inside a row
                    for (uint32_t r = 0; r < n_rows; r++) {
                        int64_t so = (int64_t)r * d->s0, doff = (int64_t)r * d->d0;
                        if (!fast) { generic_row(T, d->lin + r, &so, &doff); so += d->dst_rel; }
                        const uint32_t a = (uint32_t)((uintptr_t)(d->src + so) & 15u);
                        store_row(dp + doff, slot + r * pitch + 16u + a, n, (uint32_t)lane);
                    }
                }
            }
            bulk_commit();                                    // one group per tile, empty when registers stored it
            __syncwarp();                                     // every lane has read the slot ...
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // ... before the copy engine may overwrite it
            if (++st_slot == stages) { st_slot = 0; st_parity ^= 1u; }
        }
    }
    pdl_launch_dependents();
    bulk_wait_read(0);                                        // shared memory must outlive the stores' reads
}

// ------------------------------------------------------------------------------------------------
// host-side launchers

static thread_local int64_t g_launches = 0;
int64_t launch_count() { return g_launches; }

// the first n pointers of each side in a 256-byte parameter
static RsPtrTableT<RS_PTRS_SMALL> small_table(const RsPtrTable &ptrs) {
    RsPtrTableT<RS_PTRS_SMALL> t;
    for (int i = 0; i < RS_PTRS_SMALL; i++) { t.src[i] = ptrs.src[i]; t.dst[i] = ptrs.dst[i]; }
    return t;
}

static cudaError_t launched(cudaError_t e) {
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) ++g_launches;
    return e;
}

// every launch carries the programmatic-stream-serialization attribute unless the plan switched it off
template <typename... KArgs, typename... Args>
static cudaError_t launch_k(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t st, bool pdl, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return launched(cudaLaunchKernelEx(&cfg, kernel, args...));
}

cudaError_t launch_lsu(const RsOpDev &op, const RsPtrTable &ptrs, bool small, bool generic, int grid, bool pdl, cudaStream_t st) {
    constexpr int U = RS_LSU_UNROLL / 2;                       // 64 B in flight per thread
    if (generic) {
        if (small) return launch_k(rs_copy_lsu<uint4, U, RS_PTRS_SMALL, true>, grid, RS_LSU_THREADS, 0, st, pdl, op, small_table(ptrs));
        return launch_k(rs_copy_lsu<uint4, U, 128, true>, grid, RS_LSU_THREADS, 0, st, pdl, op, ptrs);
    }
    if (small) return launch_k(rs_copy_lsu<uint4, U, RS_PTRS_SMALL, false>, grid, RS_LSU_THREADS, 0, st, pdl, op, small_table(ptrs));
    return launch_k(rs_copy_lsu<uint4, U, 128, false>, grid, RS_LSU_THREADS, 0, st, pdl, op, ptrs);
}

// Layouts that are not 16-byte aligned AND made of short rows: the register kernel at the layout's own vector width (8, 4, 2 or 1 bytes)
// instead of the shift kernel -- assembling 16-byte windows pays when rows are long; on rows of tens of bytes most windows are partial.
template <typename V>
static cudaError_t launch_narrow_t(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, bool pdl, cudaStream_t st) {
    constexpr int U = sizeof(V) >= 8 ? 4 : 8;
    if (small) return launch_k(rs_copy_lsu<V, U, RS_PTRS_SMALL, true>, grid, RS_LSU_THREADS, 0, st, pdl, op, small_table(ptrs));
    return launch_k(rs_copy_lsu<V, U, 128, true>, grid, RS_LSU_THREADS, 0, st, pdl, op, ptrs);
}

cudaError_t launch_narrow(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int vec_bytes, int grid, bool pdl, cudaStream_t st) {
    switch (vec_bytes) {
        case 8: return launch_narrow_t<uint2>(op, ptrs, small, grid, pdl, st);
        case 4: return launch_narrow_t<uint32_t>(op, ptrs, small, grid, pdl, st);
        case 2: return launch_narrow_t<uint16_t>(op, ptrs, small, grid, pdl, st);
        default: return launch_narrow_t<uint8_t>(op, ptrs, small, grid, pdl, st);
    }
}

cudaError_t launch_shift(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, bool pdl, cudaStream_t st) {
    if (small) return launch_k(rs_copy_shift<4, RS_PTRS_SMALL>, grid, RS_LSU_THREADS, 0, st, pdl, op, small_table(ptrs));
    return launch_k(rs_copy_shift<4, 128>, grid, RS_LSU_THREADS, 0, st, pdl, op, ptrs);
}

cudaError_t prepare_bulk(int smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(rs_copy_bulk<RS_PTRS_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rs_copy_bulk<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rs_copy_tmap, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rs_copy_bulk_shift<RS_PTRS_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(rs_copy_bulk_shift<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    return e;
}

cudaError_t launch_bulk_shift(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, int block, int smem_bytes,
                              int stages, int lookahead, uint32_t stage_bytes, int mode, float pace, int burst, bool pdl, cudaStream_t st) {
    if (small) return launch_k(rs_copy_bulk_shift<RS_PTRS_SMALL>, grid, block, (size_t)smem_bytes, st, pdl, op, small_table(ptrs), stages, lookahead, stage_bytes, mode, pace, burst);
    return launch_k(rs_copy_bulk_shift<128>, grid, block, (size_t)smem_bytes, st, pdl, op, ptrs, stages, lookahead, stage_bytes, mode, pace, burst);
}

cudaError_t launch_tmap(const RsOpDev &op, const RsPtrTable &ptrs, const void *tmaps, int grid, int block, int smem_bytes, int stages,
                        int lookahead, uint32_t stage_bytes, float pace, int burst, bool pdl, cudaStream_t st) {
    static_assert(sizeof(RsTmapTable) == RS_TMAP_TABLE_BYTES, "kernels.h and the tensor-map table disagree");
    RsTmapTable tm;
    memcpy(&tm, tmaps, sizeof(tm));
    return launch_k(rs_copy_tmap, grid, block, (size_t)smem_bytes, st, pdl, op, small_table(ptrs), tm, stages, lookahead, stage_bytes, pace, burst);
}

// ------------------------------------------------------------------------------------------------
// reshard_execute_static (api.cu): the task tables of ONE launch in a file-scope array instead of the plan's cudaMalloc
// block, for callers that cannot call cudaMalloc.  Every GPU that loads the library holds these RS_STATIC_TABLE_BYTES until
// exit.  In host code the array's name is a host-side stand-in, NOT a device address: its device address is taken with
// cudaGetSymbolAddress, once per device, with that device current, and handed to the kernels as their table pointer.
static __device__ __align__(256) unsigned char g_static_tables[RS_STATIC_TABLE_BYTES];

cudaError_t static_tables(void **ptr) {                       // the array on the CURRENT device
    static std::mutex mu;
    static void *cache[64];
    *ptr = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && cache[dev]) { *ptr = cache[dev]; return cudaSuccess; }
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_tables);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) cache[dev] = p;
    *ptr = p;
    return cudaSuccess;
}

cudaError_t launch_bulk(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, int block, int smem_bytes, int stages,
                        int lookahead, uint32_t stage_bytes, float pace, int burst, bool pdl, cudaStream_t st) {
    if (small) return launch_k(rs_copy_bulk<RS_PTRS_SMALL>, grid, block, (size_t)smem_bytes, st, pdl, op, small_table(ptrs), stages, lookahead, stage_bytes, pace, burst);
    return launch_k(rs_copy_bulk<128>, grid, block, (size_t)smem_bytes, st, pdl, op, ptrs, stages, lookahead, stage_bytes, pace, burst);
}

}  // namespace rs

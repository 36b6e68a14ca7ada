// config.h -- launch-shape defaults of the executors, every one from a measurement on B200 (S3, profiles/).
// Tests and sweeps override them per plan through rs_plan_opts.tuning (include/reshard.h rs_tuning); the library reads
// no environment variable.
#pragma once

// register path: 128-bit ld.global -> st.global x k
#define RS_LSU_THREADS       256
#define RS_LSU_CTAS_PER_SM   4          // most persistent CTAs per SM (grid = SMs * CTAs per SM); every warp is a worker
#define RS_LSU_CTAS_DEFAULT  2          // CTAs per SM actually launched (more bytes in flight is slower on B200)
#define RS_LSU_CTAS_MCAST    1          // ... for large write-heavy operations (the register path has no pacing: 128-byte rows, 1 + 4 GiB: 5.05 TB/s
                                        // with 1 CTA per SM, 4.64 with 2, 4.59 with 4; AUTO sends them through tensor maps when it can: 6.09)
#define RS_LSU_CTAS_SMALL    4          // ... for operations moving <= RS_SMALL_OP_BYTES (ramp-bound, not DRAM-bound)
#define RS_LSU_TILE_BYTES    16384
#define RS_LSU_UNROLL        8          // independent vector loads in flight per thread
#define RS_LSU_TABLE_BYTES   12288      // tables (tasks + destinations + segments) up to this size are staged in shared memory at
                                        // kernel start: ONE global latency instead of a chain of dependent ones before the first load
                                        // (small operations are ramp-bound)

// TMA path: cp.async.bulk global -> shared ring -> global x k; every warp is its own pipeline
#define RS_BULK_WARPS        2          // warps (independent pipelines) per CTA, one CTA per SM
#define RS_BULK_STAGES       4          // ring slots per warp
#define RS_BULK_LOOKAHEAD    2          // loads in flight per warp before the first store is issued
#define RS_BULK_TILE_BYTES   12288      // bytes per ring slot
#define RS_BULK_SHORT_RUN    2048       // runs up to this long: many copies per tile, use the SHORT shape (4 warps x 8 KiB) -- write-heavy operations,
                                        // 1 : 1 ones under 128 MiB and tensor-map copies; larger 1 : 1 operations have a shape of their own (WIDE_11 below)
#define RS_BULK_VERY_SHORT_RUN 512      // large operations made of rows up to this long (24+ copies per 12 KiB): 8 warps x 4 slots x 6 KiB (tables.cpp many_copies)
#define RS_BULK_TILE_BYTES_MANY 6144
#define RS_BULK_MIN_FILL     0.7        // slots less full than this on average: the SHORT shape too
#define RS_BULK_TINY_FILL    0.3        // slots less than 30 % full (tiles under ~3.5 KiB): 8 warps x 3 slots x 4 KiB
#define RS_BULK_WARPS_SHORT  4
#define RS_BULK_TILE_BYTES_SHORT 8192
#define RS_BULK_CTAS_DEN       148    // CTA counts below are out of 148 SMs
#define RS_BULK_CTAS_LONG_NUM  132    // large 1 : 1 operations (WIDE_11)
// Rate matching of write-heavy (multicast) operations: every SM runs, every warp paces its tiles so that the launch
// offers this many permille of the DRAM peak (2 x memory clock x bus width = 7 672 GB/s on B200).  Measured
// (profiles/r02_pacing.md): achieved = 0.99 x offered up to 860 permille (6.52 TB/s on 1 + 8), collapse from 880 on
// (6.09, then 5.56 at 920; unpaced 5.66); runs of 512 B: up to 820 (6.18 TB/s), 6.00 at 840 -- on an IDLE chip.  The defaults below sit
// 3-5 % lower, where a chip hot from GEMMs still holds them (profiles/r02_pacing.md part 4).
#define RS_PACE_BLOCK_NS       1500           // a ring slot still being read this long after the warp asked for it: HBM is behind, back off
#define RS_PACE_BURST          2              // tiles of credit of the token bucket
#define RS_PACE_PERMILLE       825            // (850 is the best on a cold chip: 6.45 TB/s against 6.26; after GEMM bursts -- the chip power-limited, HBM hot -- the
                                              //  edge lies 3-5 % lower: 850 then gives an erratic 5.8-6.4, 825 a steady 6.25: profiles/r02_pacing.md part 4)
#define RS_PACE_PERMILLE_SHORT 775            // (cold: 6.08 TB/s at 810, 5.83 at 775; hot: 4.63 at 810, 5.85 at 775)
#define RS_PACE_PERMILLE_SHORT_DENSE 820   // short rows that are adjacent in the receivers (one bulk store per tile)
#define RS_PACE_MIN_BYTES      (64ll << 20)   // 4 + 32 MiB: 8.75 us unpaced, 9.26 paced; 16 + 128 MiB: 27.3 unpaced, 26.4 paced
#define RS_PACE_PERMILLE_WIDE_11 860          // 1 : 1 operations moving >= RS_WIDE_11_MIN_BYTES through rs_copy_bulk: 4 warps x 12 KiB per SM, paced (tables.cpp WIDE_11).
                                              //   Idle, 132 CTAs: +1 % per 10 permille up to 900 (c4 6.42 TB/s at 860, 6.48 at 870, 6.56 at 880, 6.62 at 890), collapse beyond; after GEMM
                                              //   bursts three boxes held 880 (6.41-6.57) and a fourth, whose idle rates are 1-2 % lower too, fell to 5.94-6.08 at 880 and held 6.37-6.41
                                              //   at 865, 6.26-6.39 at 850 (profiles/r02_pacing.md part 5)
#define RS_PACE_PERMILLE_11    880            // smaller 1 : 1 operations made of runs >= RS_PACE_11_MIN_RUN (2 warps on every SM; ramp-bound, far from the edge)
#define RS_PACE_PERMILLE_11_SHORT 860         // ... through tensor maps (rows of 64 B - 2 KiB)
#define RS_PACE_11_MIN_BYTES   (128ll << 20)
#define RS_WIDE_11_MIN_BYTES   (384ll << 20)  // (CUDA graphs of 50+ launches.  64 + 64 MiB of long runs: 21.9 us on 2 unpaced warps x 148 CTAs, 24.1 as WIDE_11; 128 + 128 MiB: long runs
                                              //  6.42 TB/s on 2 warps @ 880 x 148 CTAs against 6.16 as WIDE_11, config 2's pack (2 KiB rows) 6.16 on 4 x 8 KiB @ 860 against 5.86;
                                              //  256 + 256 MiB: WIDE_11 +3-5 % on P1 / P4 / P6)
#define RS_PACE_11_MIN_RUN     (1ll << 20)    // below RS_WIDE_11_MIN_BYTES: 1 : 1 operations made of runs this long keep 2 warps on every SM, paced at RS_PACE_PERMILLE_11
                                              //  (64 + 64 MiB of whole-shard copies: 6.29 TB/s against 6.14 unpaced)
#define RS_MID_MCAST_BYTES     (768ll << 20)  // paced write-heavy operations moving up to this much: the 4-warp shape
#define RS_SMALL_OP_BYTES    (32ll << 20)   // AUTO: aligned operations moving no more than this take the register path
                                            // (no shared-memory carve-out, no mbarriers: 4 MiB + 4 MiB in 3.2 us against 6.5 us;
                                            // equal at 16 + 16 MiB; from 20 + 20 MiB on the TMA ring wins: 8.1 against 8.6 us)
#define RS_SMALL_OP_BYTES_MCAST (10ll << 20)   // ... write-heavy ones (a slice with k >= 2 receivers): up to 1 + 8 MiB
#define RS_SMALL_MCAST_BYTES   (40ll << 20)    // write-heavy operations moving up to this much: 8 warps x 3 slots x 4 KiB per SM
#define RS_BULK_WARPS_SMALL_MCAST      8       // (4 + 16 MiB: 4.8 us against 6.7 us with 2 x 4 x 12 KiB and 6.4 us in registers;
#define RS_BULK_STAGES_SMALL_MCAST     3       //  4 + 32 MiB: 7.5 us either way; from 16 + 64 MiB on the default shape)
#define RS_BULK_TILE_BYTES_SMALL_MCAST 4096
#define RS_INTERLEAVE_MAX_RUN (64 << 10)    // destination runs up to this long count as a fine interleave (tile order)
#define RS_NARROW_MAX_RUN    512        // register path, layout 8-byte aligned and no more, rows shorter than this: 8-byte vectors instead of the shift
                                        // kernel (4-byte aligned: rows under 48 bytes; 1- and 2-byte aligned: under 8 bytes; api.cu)
#define RS_SHIFT_MIN_RUN     128        // ... unaligned layouts: rs_copy_bulk_shift from rows of 128 bytes on (large operations)
#define RS_BULK_MIN_RUN      512        // AUTO picks the TMA path only if every run is at least this long
#define RS_TMAP_SHORT_MIN_RUN   64          // AUTO: operations made of rows of 64-511 bytes take the tensor-map kernel when they are past the
#define RS_TMAP_SHORT_MIN_COVER 0.9        //   small-operation size and >= 90 % of their bytes move as whole boxes (else the register path)
#define RS_TMAP_SHORT_MIN_TILE  3584        //   ... and, when 1 : 1, their tiles hold at least this much
#define RS_TMAP_MAX_BYTES    (320ll << 20)  // AUTO: tensor-map copies for short-row operations moving up to this much

// TMA loads + shifted register stores (unaligned layouts): the stores are ALU work, so more warps, smaller tiles
#define RS_SHIFT_WARPS       8          // u4 (6145-byte runs, 2-byte aligned): 8 x 2 x 8 KiB = 5.6-5.7 TB/s; 4 x 4 x 8 KiB a little more,
#define RS_SHIFT_STAGES      2          // but short rows (flat walk, ~100 instructions per 512 B) need the 8 warps
#define RS_SHIFT_TILE_BYTES  8192
#define RS_PACE_PERMILLE_SHIFT       850          // rate matching of the shifted kernel, rows >= RS_PACE_SHIFT_MIN_RUN: 1 : 1 (u4: 5.96 TB/s at 800, 6.17 at 830, 6.31 at 850, 6.29 at 860; u1 5.90 / 6.11 / 6.24 / 6.30)
#define RS_PACE_PERMILLE_SHIFT_MCAST 800          // ... write-heavy (1 + 4 of u1's rows: 5.91 TB/s at 800, 4.81 at 830 -- past the edge; unpaced 4.79)
#define RS_PACE_SHIFT_MIN_BYTES      (256ll << 20)
#define RS_PACE_SHIFT_MIN_RUN         2048
#define RS_SHIFT_LONG_RUN    4096       // rows at least this long MAY leave through bulk stores (rs_tuning.shift_mode = 2; unpaced: u4 6.12 TB/s against 5.65 from registers;
                                        // paced at 850: 6.31 against 6.10 idle, 5.3 against 5.97 after GEMM bursts, so registers are the default: api.cu)
#define RS_SHIFT_MID_RUN     1024       // rows of 1-4 KiB (stored row by row from registers)
#define RS_SHIFT_WARPS_MID   8          // u1 (2050-byte rows): 6 x 3: 5.38 TB/s, 7 x 3: 6.08, 8 x 2: 5.85, 8 x 3: 5.65
#define RS_SHIFT_STAGES_MID  2          // (idle chip: 7 x 3 is best, 6.08 TB/s against 5.86-5.92; after GEMM bursts 7 x 3 falls to 4.34, 8 x 2 holds 4.92-4.97)
#define RS_SHIFT_WARPS_LONG  8          // rows >= 4 KiB: bodies realigned in the ring and stored with bulk copies.  One warp per
#define RS_SHIFT_STAGES_LONG 2          // scheduler hides no latency (~520 instructions per tile at ~6 cycles each), so many warps:
                                        // u4 4 x 4: 4.4 TB/s, 5 x 4: 5.4, 6 x 3: 6.12, 7 x 3: 6.05, 8 x 3: 5.75 (register stores, 4 x 4: 5.79) on an idle chip;
                                        // after GEMM bursts (SM clock ~1.4 GHz) 6 x 3 falls to 4.49 while 8 x 2 holds 5.69 (idle: 5.72), so 8 x 2

#define RS_BULK_DESC_BYTES   4096       // per-warp descriptor ring: 64 tiles x 64 bytes

// reshard_execute_host: pipeline over slabs of tensor dim 0
#define RS_HOST_SLABS_MAX        16
#define RS_HOST_SLAB_MIN_BYTES  (8 << 20)

#define RS_SPAN_TILE_MIN_BYTES 1024      // spans of the innermost row dim holding at least this much become one FAST tile each
#define RS_TILES_PER_WORKER   4          // small operations: tiles shrink until every warp has this many (tail balance)
#define RS_SMEM_MAX          (227 * 1024)
#define RS_STATIC_TABLE_BYTES (256 * 1024) // reshard_execute_static: the file-scope device array that holds one launch's tables (~1000 unit tasks)
#define RS_RING_MIN_SMEM_FROM (384ll << 20) // ... for operations moving at least this much (below, the overlap of the prologue is worth more: 64 + 64 MiB pack 22.4 -> 23.3 us without it)
#define RS_RING_MIN_SMEM     (116 * 1024) // ring kernels ask for at least this much: more than half an SM's shared memory, so two never share an SM

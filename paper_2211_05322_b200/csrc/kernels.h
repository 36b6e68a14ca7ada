// kernels.h -- launchers of the two executors (kernels.cu).  Internal header.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tables.h"

namespace rs {
// `pdl`: launch with the programmatic-stream-serialization attribute (kernels.cu).
// `small`: every buffer index of the launch is below RS_PTRS_SMALL, so the 256-byte pointer table is enough
// generic: the operation has GENERIC tiles (the other instantiation does not contain their walk)
cudaError_t launch_lsu(const RsOpDev &op, const RsPtrTable &ptrs, bool small, bool generic, int grid, bool pdl, cudaStream_t st);      // 16-byte aligned only
cudaError_t launch_shift(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, bool pdl, cudaStream_t st);
// the register kernel at vec_bytes = 8, 4, 2 or 1 (unaligned layouts made of short rows)
cudaError_t launch_narrow(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int vec_bytes, int grid, bool pdl, cudaStream_t st);
cudaError_t prepare_bulk(int smem_bytes);                                             // both TMA kernels, both table sizes
// pace: nanoseconds a warp lets pass per byte of DRAM traffic of its tiles (rate matching, kernels.cu); 0 = unpaced
// burst: tiles of credit a warp that fell behind may catch up with
cudaError_t launch_bulk(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, int block, int smem_bytes, int stages,
                        int lookahead, uint32_t stage_bytes, float pace, int burst, bool pdl, cudaStream_t st);
// mode: RS_SHIFT_REG (register stores) or RS_SHIFT_BULK (bodies of long rows realigned in the ring, bulk stores)
enum { RS_SHIFT_REG = 1, RS_SHIFT_BULK = 2 };
cudaError_t launch_bulk_shift(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, int block, int smem_bytes,
                              int stages, int lookahead, uint32_t stage_bytes, int mode, float pace, int burst, bool pdl, cudaStream_t st);
// tensor-map TMA path: tmaps = RS_TMAP_TABLE_BYTES bytes, RS_TMAP_BUFS CUtensorMap per side (api.cu encodes them)
#define RS_TMAP_TABLE_BYTES (2 * RS_TMAP_BUFS * 128)
cudaError_t launch_tmap(const RsOpDev &op, const RsPtrTable &ptrs, const void *tmaps, int grid, int block, int smem_bytes, int stages,
                        int lookahead, uint32_t stage_bytes, float pace, int burst, bool pdl, cudaStream_t st);
// device address, on the current device, of the file-scope table array of reshard_execute_static (RS_STATIC_TABLE_BYTES bytes, 256-byte aligned)
cudaError_t static_tables(void **ptr);
int64_t launch_count();
}  // namespace rs

// kernels.h -- launchers of the two executors (kernels.cu).  Internal header.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tables.h"

namespace rs {
// `small`: every buffer index of the launch is below RS_PTRS_SMALL, so the 256-byte pointer table is enough
cudaError_t launch_lsu(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, cudaStream_t st);      // 16-byte aligned only
cudaError_t launch_shift(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, cudaStream_t st);
cudaError_t prepare_bulk(int smem_bytes);                                             // both TMA kernels, both table sizes
cudaError_t launch_bulk(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, int block, int smem_bytes, int stages,
                        int lookahead, uint32_t stage_bytes, cudaStream_t st);
cudaError_t launch_bulk_shift(const RsOpDev &op, const RsPtrTable &ptrs, bool small, int grid, int block, int smem_bytes,
                              int stages, int lookahead, uint32_t stage_bytes, cudaStream_t st);
int64_t launch_count();
}  // namespace rs

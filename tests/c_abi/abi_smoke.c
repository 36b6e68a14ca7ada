/* A plain C99 user of include/reshard.h: no Python, no torch, no C++.  Built and run by
 * tests/test_c_abi.py.  Host-only part: plans, queries, S3.2 schedule, S4 timeline.  With a CUDA
 * device (argv[1] = "gpu"): config 1 of BASELINE.json through reshard_execute and pack/unpack,
 * checked against the definition (value = global linear index). */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <cuda_runtime_api.h>
#include "reshard.h"

#define CHECK(x) do { rs_status s_ = (x); if (s_ != RS_OK) { fprintf(stderr, "%s:%d %s: %s (%s)\n", __FILE__, __LINE__, #x, reshard_strerror(s_), reshard_last_error()); return 1; } } while (0)

int main(int argc, char **argv) {
    const int gpu = argc > 1 && strcmp(argv[1], "gpu") == 0;
    const int64_t shape[2] = {8, 16};
    const int32_t mesh[2] = {1, 2};
    rs_plan *plan = NULL;
    rs_plan_info info;
    rs_plan_opts opts;
    memset(&opts, 0, sizeof opts);
    opts.flags = gpu ? 0 : RS_HOST_ONLY;
    opts.schedule = RS_SCHED_ENSEMBLE;
    /* config 1, prose intent (R21): rows split over 2 devices -> columns split */
    CHECK(reshard_plan_ex(shape, 2, 4, mesh, 2, "S1,R", mesh, 2, "R,S1", &opts, &plan));
    CHECK(reshard_plan_info(plan, &info));
    if (info.n_slices != 4 || info.n_src != 2 || info.n_dst != 2 || info.tensor_bytes != 512) { fprintf(stderr, "unexpected plan\n"); return 1; }
    rs_schedule_info si;
    int32_t order[4], host[4];
    int64_t start[4];
    CHECK(reshard_plan_schedule(plan, &si, host, start, order));
    if (si.makespan != 256 || si.busiest_host_bytes != 256) { fprintf(stderr, "unexpected schedule: %lld\n", (long long)si.makespan); return 1; }
    /* S4: 4 stages, 8 micro-batches, f = 1, b = 2, free communication: (M + S - 1)(f + b) = 33 */
    int64_t f[4] = {1, 1, 1, 1}, b[4] = {2, 2, 2, 2};
    rs_pipeline_opts po;
    rs_pipeline_result pr;
    memset(&po, 0, sizeof po);
    po.schedule = RS_PIPE_EAGER_1F1B; po.n_stages = 4; po.n_micro_batches = 8; po.overlap = 1; po.fwd = f; po.bwd = b;
    CHECK(reshard_pipeline_simulate(&po, &pr, NULL, NULL, NULL, NULL));
    if (pr.makespan != 33 || pr.warmup[0] != 7 || pr.peak_activations[0] != 7) { fprintf(stderr, "unexpected timeline\n"); return 1; }
    if (reshard_plan(shape, 2, 3, mesh, 2, "S1,R", mesh, 2, "R,S1", RS_HOST_ONLY, &plan) != RS_EINVAL) return 1;   /* plan untouched on failure */
    if (gpu) {
        float h_src[2][64], h_dst[2][64], *d_src[2], *d_dst[2];
        void *arena = NULL;
        int r, i, j;
        for (r = 0; r < 2; r++) {
            for (i = 0; i < 4; i++) for (j = 0; j < 16; j++) h_src[r][i * 16 + j] = (float)((r * 4 + i) * 16 + j);   /* value = global index */
            if (cudaMalloc((void **)&d_src[r], 256) || cudaMalloc((void **)&d_dst[r], 256)) return 2;
            cudaMemcpy(d_src[r], h_src[r], 256, cudaMemcpyHostToDevice);
            cudaMemset(d_dst[r], 0xFF, 256);
        }
        if (cudaMalloc(&arena, (size_t)info.arena_bytes)) return 2;
        int pass;
        for (pass = 0; pass < 2; pass++) {
            const void *src[2] = {d_src[0], d_src[1]};
            void *dst[2] = {d_dst[0], d_dst[1]};
            if (pass == 0) CHECK(reshard_execute(plan, src, dst, NULL));
            else { CHECK(reshard_pack(plan, src, arena, NULL)); CHECK(reshard_unpack(plan, arena, dst, NULL)); }
            if (cudaDeviceSynchronize() != cudaSuccess) return 2;
            for (r = 0; r < 2; r++) {
                cudaMemcpy(h_dst[r], d_dst[r], 256, cudaMemcpyDeviceToHost);
                for (i = 0; i < 8; i++) for (j = 0; j < 8; j++)
                    if (h_dst[r][i * 8 + j] != (float)(i * 16 + r * 8 + j)) { fprintf(stderr, "pass %d: device %d element (%d,%d) wrong\n", pass, r, i, j); return 1; }
                cudaMemset(d_dst[r], 0xFF, 256);
            }
        }
        if (reshard_launch_count() != 3) return 1;
    }
    reshard_plan_destroy(plan);
    printf("c abi ok (%s, %s)\n", gpu ? "gpu" : "host only", reshard_version());
    return 0;
}

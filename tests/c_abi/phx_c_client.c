/*
 * phx_c_client.c — a plain C99 program that drives the hot path through include/phx.h alone: no Python,
 * no torch, buffers from cudaMalloc / cudaHostAlloc.  Test infrastructure (tests/test_gpu_c_abi.py builds
 * and runs it): it reads the initial p and the gradients of each step from files, runs
 *     create -> bind -> set_state -> [step_and_snapshot -> flush_async] x steps -> wait
 *     -> (in-flight step) -> zero the live shard -> restore -> recompute the in-flight step
 *     -> the gradient producer's epilogue (phx_grads_finalize_async) feeding one step
 *     -> two steps through the graph-capturable form (phx_graph_begin / flush / step / end), called eagerly
 *     -> a second fault recovered in two phases (phx_restore_async / phx_restore_wait_params) and one more step
 * and writes p, m, v, the bf16 copy and the two host replica slots to an output file that the test
 * compares byte for byte with the CPU oracle.
 *
 * usage: phx_c_client <in.bin> <out.bin>
 *   in.bin : u64 n_tensors, u64 numel[n_tensors], u32 dp_size, u32 dp_rank, u32 steps, f32 max_grad_norm,
 *            u64 chunk_bytes, f32 p0[n_padded], then (steps + 1) x bf16 g[n_padded], f32 scale, f32 g32[n_padded]
 *   out.bin: u64 n_padded, u64 restored_step, f32 p, m, v [n_padded] each, u16 p16[n_padded],
 *            u8 replica[2 * slot_stride]
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "phx.h"

#define CK(call)                                                                              \
    do {                                                                                      \
        int rc_ = (call);                                                                     \
        if (rc_ != PHX_OK) {                                                                  \
            fprintf(stderr, "%s -> %d (%s)\n", #call, rc_, phx_strerror(rc_));                \
            return 2;                                                                         \
        }                                                                                     \
    } while (0)
#define CU(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess) {                                                              \
            fprintf(stderr, "%s -> %s\n", #call, cudaGetErrorString(e_));                     \
            return 3;                                                                         \
        }                                                                                     \
    } while (0)

static int rd(FILE *f, void *dst, size_t n) { return fread(dst, 1, n, f) == n ? 0 : -1; }

int main(int argc, char **argv)
{
    if (argc != 3) return 1;
    FILE *in = fopen(argv[1], "rb");
    if (!in) return 1;
    uint64_t nt, chunk;
    uint32_t dp_size, dp_rank, steps;
    float max_norm;
    if (rd(in, &nt, 8)) return 1;
    phx_tensor_desc_t *layout = (phx_tensor_desc_t *)calloc(nt, sizeof(*layout));
    for (uint64_t i = 0; i < nt; ++i) {
        if (rd(in, &layout[i].numel, 8)) return 1;
        layout[i].tensor_id = (uint32_t)i;
    }
    if (rd(in, &dp_size, 4) || rd(in, &dp_rank, 4) || rd(in, &steps, 4) || rd(in, &max_norm, 4) || rd(in, &chunk, 8))
        return 1;

    phx_config_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.chunk_bytes = chunk;
    cfg.max_grad_norm = max_norm;
    phx_shard_t *s = NULL;
    CK(phx_shard_create(layout, (size_t)nt, dp_size, dp_rank, &cfg, &s));
    phx_shard_info_t info;
    CK(phx_shard_info(s, &info));
    const uint64_t N = info.n_padded;

    float *d_p, *d_m, *d_v;
    void *d_p16, *d_staging, *h_replica, *d_g;
    cudaStream_t compute, side;
    CU(cudaMalloc((void **)&d_p, 4 * N));
    CU(cudaMalloc((void **)&d_m, 4 * N));
    CU(cudaMalloc((void **)&d_v, 4 * N));
    CU(cudaMalloc(&d_p16, 2 * N));
    CU(cudaMalloc(&d_g, 2 * N));
    CU(cudaMalloc(&d_staging, info.staging_depth * info.slot_stride));
    CU(cudaHostAlloc(&h_replica, 2 * info.host_slot_stride, cudaHostAllocMapped));
    memset(h_replica, 0, 2 * info.host_slot_stride);
    CU(cudaStreamCreate(&compute));
    CU(cudaStreamCreate(&side));

    float *h_f = (float *)malloc(4 * N);
    uint16_t *h_g = (uint16_t *)malloc(2 * N * (steps + 1));
    float scale = 1.0f;
    float *h_g32 = (float *)malloc(4 * N);
    if (rd(in, h_f, 4 * N) || rd(in, h_g, 2 * N * (steps + 1)) || rd(in, &scale, 4) || rd(in, h_g32, 4 * N)) return 1;
    fclose(in);
    CU(cudaMemcpy(d_p, h_f, 4 * N, cudaMemcpyHostToDevice));
    CU(cudaMemset(d_m, 0, 4 * N));
    CU(cudaMemset(d_v, 0, 4 * N));

    CK(phx_shard_bind(s, d_p, d_m, d_v, d_p16, d_staging, h_replica));
    CK(phx_shard_set_state(s, 0, compute));
    const char blob[] = "rng-state-of-the-c-client";
    CK(phx_set_user_metadata(s, blob, (uint32_t)sizeof(blob)));

    const float lr = 3e-4f, b1 = 0.9f, b2 = 0.95f, eps = 1e-8f, wd = 0.1f;
    for (uint32_t t = 1; t <= steps; ++t) {
        CU(cudaMemcpyAsync(d_g, h_g + (size_t)(t - 1) * N, 2 * N, cudaMemcpyHostToDevice, compute));
        CK(phx_step_and_snapshot(s, d_g, lr, b1, b2, eps, wd, t, compute));
        CK(phx_snapshot_flush_async(s, side));
    }
    CK(phx_snapshot_wait(s, steps));
    /* the in-flight step: launched, then the live shard is lost */
    CU(cudaMemcpyAsync(d_g, h_g + (size_t)steps * N, 2 * N, cudaMemcpyHostToDevice, compute));
    CK(phx_step_and_snapshot(s, d_g, lr, b1, b2, eps, wd, steps + 1, compute));
    CU(cudaStreamSynchronize(compute));
    CU(cudaMemset(d_p, 0, 4 * N));
    CU(cudaMemset(d_m, 0, 4 * N));
    CU(cudaMemset(d_v, 0, 4 * N));
    CU(cudaMemset(d_p16, 0, 2 * N));
    CU(cudaMemset(d_staging, 0xA5, info.staging_depth * info.slot_stride));
    uint64_t back = 0;
    CK(phx_restore(s, compute, &back));
    char got[128];
    uint32_t glen = 0;
    CK(phx_restored_user_metadata(s, got, sizeof(got), &glen));
    if (glen != sizeof(blob) || memcmp(got, blob, glen) != 0) {
        fprintf(stderr, "user metadata did not come back\n");
        return 4;
    }
    /* recompute of the in-flight step ("at most one step of re-execution") */
    CK(phx_step_and_snapshot(s, d_g, lr, b1, b2, eps, wd, back + 1, compute));
    CK(phx_snapshot_flush_async(s, side));

    /* SURVEY 8(f4), second half: the gradients of the next step come out of the producer's epilogue (fp32 main
     * gradients x scale -> bf16 + sum of squares, one pass); the step then needs no pass of its own over them */
    float *d_g32;
    double *d_sum;
    CU(cudaMalloc((void **)&d_g32, 4 * N));
    CU(cudaMalloc((void **)&d_sum, 8));
    CU(cudaMemcpyAsync(d_g32, h_g32, 4 * N, cudaMemcpyHostToDevice, compute));
    CK(phx_grads_finalize_async(s, d_g32, scale, d_g, d_sum, compute));
    if (max_norm > 0.0f) CK(phx_set_clip_partials(s, d_sum, 1));
    CK(phx_step_and_snapshot(s, d_g, lr, b1, b2, eps, wd, back + 2, compute));

    /* the graph-capturable form, called eagerly: flush of the pending snapshot, then step, twice */
    void *d_ga, *d_gb;
    CU(cudaMalloc(&d_ga, 2 * N));
    CU(cudaMalloc(&d_gb, 2 * N));
    CU(cudaMemcpyAsync(d_ga, h_g, 2 * N, cudaMemcpyHostToDevice, compute));
    CU(cudaMemcpyAsync(d_gb, h_g + N, 2 * N, cudaMemcpyHostToDevice, compute));
    CK(phx_graph_begin(s, lr, b1, b2, eps, wd, compute));
    CK(phx_graph_flush_async(s, side));
    CK(phx_graph_step_and_snapshot(s, d_ga, compute));
    CK(phx_graph_flush_async(s, side));
    CK(phx_graph_step_and_snapshot(s, d_gb, compute));
    uint64_t last = 0;
    CK(phx_graph_end(s, &last));
    if (last != back + 4) {
        fprintf(stderr, "graph form ended at step %llu, expected %llu\n", (unsigned long long)last, (unsigned long long)(back + 4));
        return 5;
    }
    /* a second fault, recovered in TWO PHASES (phx_restore_async): the newest snapshot is flushed, the live shard is
     * lost, the parameters come back first on the side stream, the compute stream waits for them only, and the next
     * step waits for the moments by itself */
    CK(phx_snapshot_flush_async(s, side));
    CK(phx_snapshot_wait(s, last));
    CU(cudaStreamSynchronize(compute));
    CU(cudaMemset(d_p, 0, 4 * N));
    CU(cudaMemset(d_m, 0, 4 * N));
    CU(cudaMemset(d_v, 0, 4 * N));
    CU(cudaMemset(d_p16, 0, 2 * N));
    uint64_t back2 = 0;
    CK(phx_restore_async(s, side, &back2));
    CK(phx_restore_wait_params(s, compute));
    if (back2 != last) {
        fprintf(stderr, "two-phase restore came back at step %llu, expected %llu\n", (unsigned long long)back2, (unsigned long long)last);
        return 6;
    }
    CK(phx_step_and_snapshot(s, d_ga, lr, b1, b2, eps, wd, back2 + 1, compute));
    CU(cudaStreamSynchronize(compute));
    CU(cudaStreamSynchronize(side));

    FILE *out = fopen(argv[2], "wb");
    if (!out) return 1;
    fwrite(&N, 8, 1, out);
    fwrite(&back, 8, 1, out);
    float *planes[3];
    planes[0] = d_p;
    planes[1] = d_m;
    planes[2] = d_v;
    for (int k = 0; k < 3; ++k) {
        CU(cudaMemcpy(h_f, planes[k], 4 * N, cudaMemcpyDeviceToHost));
        fwrite(h_f, 4, N, out);
    }
    CU(cudaMemcpy(h_f, d_p16, 2 * N, cudaMemcpyDeviceToHost));
    fwrite(h_f, 2, N, out);
    fwrite(h_replica, 1, 2 * info.host_slot_stride, out);
    fclose(out);

    uint64_t launches = 0;
    CK(phx_kernel_launches(s, &launches));
    printf("phx_c_client ok: n_padded=%llu restored_step=%llu kernel_launches=%llu\n", (unsigned long long)N,
           (unsigned long long)back, (unsigned long long)launches);
    CK(phx_shard_destroy(s));
    return 0;
}

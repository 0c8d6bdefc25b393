/*
 * phx_probe.h — BENCH-ONLY diagnostic, NOT part of the product boundary (include/phx.h is).
 * Built into its own library (libphx_probe.so) so that the product library exports product calls only.
 *
 * phx_hbm_probe_async: enqueue ONE streaming pass over n_read planes that are read and n_write planes that
 * are written (plane i at d_buf + i*plane_bytes, reads first; d_buf: device memory of
 * (n_read+n_write)*plane_bytes bytes, 256-byte aligned; plane_bytes a multiple of 256; each count <= 8) with
 * the fused step's access pattern (one 256-bit vector per thread and plane, same cache hints, 256-thread
 * CTAs) and no arithmetic — the HBM ceiling for that read:write mix, the context bench.py prints next to
 * the driver-measured copy peak.  The written planes are overwritten with junk.
 * Returns 0, -1 (invalid argument), -2 (alignment) or -9 (CUDA error).
 */
#ifndef PHX_PROBE_H
#define PHX_PROBE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
__attribute__((visibility("default"))) int phx_hbm_probe_async(void *d_buf, uint64_t plane_bytes, uint32_t n_read,
                                                               uint32_t n_write, void *stream);
/* The same pass with a PERSISTENT structure: `grid` CTAs of 256 threads walking the groups with a grid stride
 * (e.g. 148 x 4) instead of one short-lived CTA per 256 groups — the structural alternative the fused step was
 * measured against (profiles/r02_structure_probe.md). */
__attribute__((visibility("default"))) int phx_hbm_probe_persistent_async(void *d_buf, uint64_t plane_bytes, uint32_t n_read,
                                                                          uint32_t n_write, uint32_t grid, void *stream);
#ifdef __cplusplus
}
#endif
#endif

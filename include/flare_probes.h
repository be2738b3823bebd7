/*
 * flare_probes.h -- BENCH HOOKS, not part of the product ABI (include/flare_b200.h): three small device probes
 * that bench.py uses as roofline denominators where MEASURED_PEAKS.json has no entry (it carries an HBM copy and
 * bf16 GEMM figure only; this path computes in FP64).  Built as a separate library, libflare_probes.so, from
 * paper_2204_12573_b200/csrc/probes.cu; the force-field library neither links nor calls it.
 *
 * Each probe allocates its own scratch with cudaMalloc, runs on the legacy default stream of `cuda_device`,
 * synchronises, frees, and returns the best of a few timed launches (CUDA events); a negative value = CUDA error.
 */
#ifndef FLARE_PROBES_H
#define FLARE_PROBES_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* FP64 tensor-pipe issue peak in TFLOP/s: register-resident mma.sync.m8n8k4.f64 loop, 8 independent
   accumulator pairs per warp, 8 warps per CTA, 2 CTAs per SM (DMMA.8x8x4 = 512 flop per warp instruction). */
double flare_probe_fp64_dmma_tflops(int cuda_device);

/* FP64 ALU peak in TFLOP/s: register-resident chains of independent DFMAs (2 flop per lane per instruction),
   8 chains per thread, 8 warps per CTA, 4 CTAs per SM. */
double flare_probe_fp64_dfma_tflops(int cuda_device);

/* HBM copy bandwidth in GB/s (read + write bytes) of a grid-stride 16-byte copy over `bytes` bytes per buffer
   (use a size far above the 126 MB L2); the cross-check of MEASURED_PEAKS.json's hbm_gbs. */
double flare_probe_hbm_copy_gbs(int cuda_device, size_t bytes);

#ifdef __cplusplus
}
#endif
#endif /* FLARE_PROBES_H */

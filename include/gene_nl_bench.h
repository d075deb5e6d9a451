/*
 * gene_nl_bench.h -- BENCHMARK-ONLY entry points of libgene_nl.so.  Not part of the product boundary
 * (include/gene_nl.h): nothing on the hot path calls them; bench.py uses them for the per-kernel rooflines and
 * for the measured FP64 / shared-memory denominators (SURVEY.md 8(d) asks for a measured FP64 peak).
 */
#ifndef GENE_NL_BENCH_H
#define GENE_NL_BENCH_H

#include "gene_nl.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * gene_nl_compute_profiled -- gene_nl_compute with a CUDA-event pair recorded on `stream` around every
 * kernel launch, then a stream synchronise.  ms[c] receives the summed device time [ms] and
 * launches[c] the launch count of kernel class c (arrays of GENE_NL_KERNEL_CLASSES entries):
 *   0 k_xinv       x-synthesis: derivative + pad + x half of the transform to real space
 *   1 k_yreal      chi real-space fields (dx chi, dy chi)
 *   2 k_ybracket   y-synthesis + bracket + y-analysis           (batched path, large planes)
 *   3 k_xfwd       x-analysis + delete modes + prefactor + add  (batched path, large planes)
 *   4 k_plane_fused  the whole g-side of a plane in one persistent kernel, x<->y hand-over in shared
 *                  memory (one SM, or a thread-block cluster for planes that exceed it)
 */
#define GENE_NL_KERNEL_CLASSES 5
int gene_nl_compute_profiled(gene_nl_plan* h, const void* chi, const void* g, void* rhs, double scale,
                             void* stream, double* ms, int* launches);

/*
 * gene_nl_probe_peaks -- micro-benchmarks of the two units that bound this path, on the current device.
 * out[0] = FP64 DFMA throughput [TFLOP/s] from independent register-resident FMA chains on all SMs;
 * out[1] = shared-memory bandwidth [GB/s] from conflict-free 128-bit loads+stores on all SMs;
 * out[2] = SM clock [MHz] reported by the driver at the end of the probe.  Returns 0 on success.
 */
int gene_nl_probe_peaks(double* out3);

/*
 * gene_nl_probe_exchange -- the exchange of complex128 values between the lanes of a warp (the step between two
 * register-resident FFT stages) next to the FP64 work of one radix-8 butterfly per 8 values.  With 8 warps per SM:
 * out[0] = ns per iteration for the FMAs alone, out[1] = with the exchange through a per-warp shared-memory tile
 * (8 STS.128 + 8 LDS.128 per lane), out[2] = with the exchange by warp shuffles (32 SHFL per lane); out[3..5] = the same
 * with 16 warps per SM, per 8 warps; out[6..8] = the same with 8 warps per SM and twice the FP64 work per exchange (tells
 * a shared-memory bandwidth bound from a serialisation of the two pipes).  SURVEY.md sect. 7 asked for this measurement before relying on "warp-shuffle
 * butterflies" (north_star); DESIGN.md sect. 6h has the result.
 */
int gene_nl_probe_exchange(double* out9);

#ifdef __cplusplus
}
#endif
#endif /* GENE_NL_BENCH_H */

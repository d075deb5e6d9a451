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

#ifdef __cplusplus
}
#endif
#endif /* GENE_NL_BENCH_H */

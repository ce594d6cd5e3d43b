/*
 * ris_bench.h -- measurement and diagnostic entry points of libris_b200.so.  NOT part of the product boundary
 * (include/ris.h): bench.py uses the peak probes as roofline denominators, the -m gpu tests use the layout queries to
 * aim their sampled outputs at tile edges.  Nothing here touches the hot path's results.
 */
#ifndef RIS_BENCH_H
#define RIS_BENCH_H

#include "ris.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Runs an independent-DFMA-chain kernel on every SM and returns the achieved FP64 rate in TFLOP/s (the denominator
 * of the "% FP64 peak" figure of BASELINE.json's metric; MEASURED_PEAKS.json carries no FP64 number).
 * cuda_stream: a cudaStream_t.  RIS_ECUDA on failure. */
int ris_probe_fp64_peak(double* tflops, void* cuda_stream);
/* Same for the FP64 tensor path: independent mma.sync.m8n8k4.f64 chains (the denominator for the Gamma^P GEMMs of
 * Eqs. 32-34, 39). */
int ris_probe_fp64_mma_peak(double* tflops, void* cuda_stream);

/* Layout of the pair-restricted Gamma^P GEMM-2: the spatial position of every AO
 * (ao_pos_host[nao], host pointer, filled by the call) and the tile geometry: gathered partner rows of a tile
 * (panel_rows), aux functions of a tile (tile_cols), number of tiles, number of partner-list entries (two per packed
 * pair element).  Any output pointer may be NULL.  RIS_EINVAL on a null context. */
int ris_diag_gemm2_layout(ris_ctx* ctx, int32_t* ao_pos_host, int* panel_rows, int* tile_cols, int* ntiles, int* nentries);

#ifdef __cplusplus
}
#endif
#endif /* RIS_BENCH_H */

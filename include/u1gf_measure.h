/* u1gf_measure.h -- measurement helpers, NOT part of the method (include/u1gf.h is the method's boundary).
 *
 * Two groups:
 *   (1) u1gf_last_launch_count, exported by libu1gf.so: how many kernels of that library the calling thread's most
 *       recent compute call launched.  Exact for the library's own kernels; the CUB radix-sort / scan launches inside
 *       u1gf_count_copies, u1gf_paper_count and u1gf_merge_copy_tables are library code and are NOT counted.
 *   (2) roofline denominators measured on the device in use, exported by the separate libu1gf_measure.so
 *       (csrc/peaks.cu), so that no microbenchmark lives in the product library.  Error text of that library:
 *       u1gf_measure_last_error().  Same return codes as include/u1gf.h.
 *
 *   u1gf_measure_fp64_peak   runs a dependent-chain-free DFMA kernel on all SMs for about `ms` milliseconds and
 *                            returns FP64 FMA instructions (thread-level) per second in *dfma_per_s.
 *   u1gf_measure_fp64_rate   the same rate for a DFMA stream of a given operand pattern: 0 = the stream of
 *                            u1gf_measure_fp64_peak (one register operand, two constants); 1 = three distinct
 *                            register operands per DFMA; 2 = the complex multiply-accumulate pattern of the
 *                            neighbour sum w_i (Eq. 5); 3 / 4 = stream 0 / stream 1 with two independent
 *                            integer instructions per DFMA (FP64 FMAs counted only); 5 = one dependent chain per
 *                            warp, one warp per scheduler (rate = threads in flight / dependent-issue latency);
 *                            6 = FP64 tensor-core DMMA m8n8k4, 8 FMAs per thread and instruction (the same pipe as
 *                            DFMA: its rate is the pipe's, 64 lanes x SM clock).
 *   u1gf_measure_smem_rate   warp-level shared-memory instructions per second of a mix: 0 = 4 lane-strided LDS.128
 *                            + 1 STS.128 (neighbours of 32 starts and the store), 1 = 8 warp-uniform LDS.128
 *                            (links), 2 = both (the 13 shared-memory instructions of one 4^4 site update).
 *   u1gf_measure_smem_peak   same for 128-bit conflict-free shared-memory loads, bytes per second.
 *   u1gf_measure_dsmem_rate  thread-block clusters of `cluster_size` CTAs (512 threads, 200 KB of shared memory each --
 *                            the footprint of a resident relaxation kernel): bytes per second and SM that a CTA pulls
 *                            out of the shared memory of its neighbour in the cluster (remote = 1) or of its own
 *                            through the cluster window (remote = 0) with 128-bit loads, 512 bytes per warp; and how
 *                            many such clusters the device holds at once.  The halo exchange of a cluster-resident
 *                            kernel for 6^4 / 8^4 would run at this rate.
 */
#ifndef U1GF_MEASURE_H
#define U1GF_MEASURE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* libu1gf.so */
int32_t u1gf_last_launch_count(void);

/* libu1gf_measure.so */
const char* u1gf_measure_last_error(void);
int u1gf_measure_fp64_peak(double ms, double* dfma_per_s, void* cuda_stream);
int u1gf_measure_fp64_rate(int32_t pattern, double ms, double* dfma_per_s, void* cuda_stream);
int u1gf_measure_smem_peak(double ms, double* bytes_per_s, void* cuda_stream);
int u1gf_measure_smem_rate(int32_t mix, double ms, double* instr_per_s, void* cuda_stream);
int u1gf_measure_dsmem_rate(int32_t cluster_size, int32_t remote, double ms, double* bytes_per_s_per_sm,
                            int32_t* max_active_clusters, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* U1GF_MEASURE_H */

/* mf_probe.h — entry points of lib/libmorefit_b200_probe.so: measurement and test probes (mf_probe.cu).  NOT part of the
 * product's C-ABI (include/morefit_b200.h); bench.py and the GPU tests load this library beside the product.
 * Every call takes the CUDA device index and a cudaStream_t (may be NULL) and returns 0, or the cudaError_t that stopped it. */
#ifndef MF_PROBE_H
#define MF_PROBE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
/* fp64-pipe issue rate of the GPU in DFMA thread-instructions per second, measured with register-only DFMA chains
 * (nominal B200: 148 SMs x 64 lanes x 1.965 GHz = 1.86e13). */
int mfp_fp64_rate(int device, void* stream, double* dfma_per_second);
/* fp64 tensor-core (DMMA m8n8k4) rate: out4[0] = fp64 FMAs per second with DMMA alone, out4[1] = with DFMA alone,
 * out4[2] = time(4 DMMA + 8 DFMA per step) / (time of each alone, added): 1.0 means the two serialise,
 * out4[3] = the same for 1 DMMA + 8 DFMA per step. */
int mfp_dmma_rate(int device, void* stream, double* out4);
/* Read bandwidth in bytes/s of a `bytes`-sized device buffer that one kernel reads `repeats` times with 16-byte loads:
 * L2 bandwidth when bytes fits the L2 and repeats > 1, HBM otherwise. */
int mfp_read_bandwidth(int device, void* stream, size_t bytes, int repeats, double* bytes_per_second);
/* The kernels' own device math (mf_math.cuh) element by element: op 0 = mf_exp (finite x < 709; x <= -708 gives 0),
 * 1 = mf_log (positive normal x), 2 = mf_rcp, 3 = mf_exp32, the table-by-shuffle exp of the event loops (x below about
 * -708 gives a value in [2^-1022, 2^-1021], which the kernels treat as zero).  x_host, y_host: host, n doubles. */
int mfp_math(int device, void* stream, int op, int64_t n, const double* x_host, double* y_host);
#ifdef __cplusplus
}
#endif
#endif

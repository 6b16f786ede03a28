/* phoebe_elph_probes.h -- measurement aids of bench.py, exported by libphoebe_elph_probes.so (NOT by the product
 * library libphoebe_elph.so): the FP64 and HBM ceilings the roofline fractions are reported against (SURVEY.md 8(d)
 * "Peaks": no vendor figure for B200 FP64 is available, so the ceilings are measured in the same run as the kernels).
 * Error codes as in phoebe_elph.h: 0 OK, -1 null pointer, -2 bad argument, -6 CUDA error / no device. */
#ifndef PHOEBE_ELPH_PROBES_H
#define PHOEBE_ELPH_PROBES_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* FP64 ceiling probes used for the roofline denominators: runs a
 * register-resident loop of dependent-free FP64 FMAs (kind 0: DFMA, kind 1: mma.sync
 * m8n8k4 DMMA) on every SM for `iters` iterations and writes the achieved TFLOP/s.
 * Synchronises the stream.  Errors: E_NULL, E_DIMS, E_CUDA. */
int phoebe_elph_probe_fp64(int32_t kind, int32_t iters, void* cuda_stream, double* tflops_out);

/* HBM read-stream probe: sums `bytes` of DEVICE memory with 128-bit loads; writes GB/s. */
int phoebe_elph_probe_hbm_read(const void* buf_dev, size_t bytes, void* cuda_stream, double* gbs_out);

#ifdef __cplusplus
}
#endif
#endif /* PHOEBE_ELPH_PROBES_H */

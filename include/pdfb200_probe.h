/*
 * pdfb200_probe.h -- machine probes used by bench.py, in a library of their own (libpdfb200_probe.so):
 * they evaluate nothing of the method and are not part of the product library libpdfb200.so.
 */
#ifndef PDFB200_PROBE_H
#define PDFB200_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif

/*
 * pdfb_probe -- machine probes for the bounds MEASURED_PEAKS.json does not carry (SURVEY.md 8(d):
 * the FP64 peak must be measured).  Not part of the method; used by bench.py only.
 *   PDFB_PROBE_FP64  *result = FP64 fused multiply-adds per second (thread level) of independent
 *                    DFMA chains at full occupancy
 *   PDFB_PROBE_LDS   *result = bytes per second delivered by conflict-free LDS.128 from shared memory
 * Synchronous; allocates and frees its own scratch.  result: host pointer.
 * Returns 0, -1 (bad argument) or -4 (CUDA error / no device): the codes of pdfb200.h.
 */
#define PDFB_PROBE_FP64 1
#define PDFB_PROBE_LDS 2
int pdfb_probe(int which, int device, double *result);

#ifdef __cplusplus
}
#endif
#endif /* PDFB200_PROBE_H */

/*
 * lya_peaks.h -- C-ABI of liblya_peaks.so: microbenchmarks of the units that bound the pair loops
 * (DESIGN.md "Rooflines").  NOT part of the product library: only bench.py loads it, to print the
 * measured denominators beside the roofline fractions.
 */
#ifndef LYA_PEAKS_H
#define LYA_PEAKS_H
#ifdef __cplusplus
extern "C" {
#endif

/* Each kind runs on `device` (CUDA ordinal), returns operations per second through *rate (host out)
 * and synchronises.  Returns 0 on success, a cudaError_t value otherwise.
 *   LYA_PEAK_FP64_FMA     warp-level DFMA instructions x 32 lanes per second
 *   LYA_PEAK_FP64_ADD     same for DADD
 *   LYA_PEAK_SMEM_CAS64   lane-level shared-memory fp64 atomic adds (CAS loop) per second,
 *                         random bins of a 2500-entry histogram
 *   LYA_PEAK_SMEM_ADD32   lane-level native shared-memory u32 atomic adds per second
 *   LYA_PEAK_L2_RED64     lane-level red.global.add.f64 per second into an L2-resident
 *                         2500 x 2500 double matrix (random row, contiguous segment)
 *   LYA_PEAK_L2_RED64_SCATTER  the same with every lane on its own random element of a 19 MB
 *                         array (the triangle-bin accumulators of lya_xi3pcf) */
typedef enum {
    LYA_PEAK_FP64_FMA = 0, LYA_PEAK_FP64_ADD = 1, LYA_PEAK_SMEM_CAS64 = 2,
    LYA_PEAK_SMEM_ADD32 = 3, LYA_PEAK_L2_RED64 = 4, LYA_PEAK_L2_RED64_SCATTER = 5
} lya_peak_kind;
int lya_measure_peak(int device, lya_peak_kind kind, double *rate);

#ifdef __cplusplus
}
#endif
#endif /* LYA_PEAKS_H */

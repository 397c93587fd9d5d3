/* hard_probe.h — measurement utility, NOT part of the product ABI (include/hard.h) and not on the hot path.
 * Built as its own shared library, paper_2509_08971_b200/libhard_probe.so, by the same build step; bench.py
 * loads it for the roofline denominator.  SURVEY.md Finding 2 / BASELINE.md §2: the fused stage kernel is
 * bound by the fp64 pipe and MEASURED_PEAKS.json has no fp64 entry, so the fp64 vector peak is measured live.
 */
#ifndef HARD_B200_HARD_PROBE_H
#define HARD_B200_HARD_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif

/* fp64 vector peak of the current CUDA device in TFLOP/s: register-resident chains of independent DFMA on all
 * SMs, best of 4 timed launches (one DFMA = 2 flop).  The second argument is reserved (may be NULL).
 * Returns 0 on success, -1 bad argument, -2 CUDA error, -3 out of memory (the HARD_* codes of hard.h). */
int hard_probe_fp64_peak(double* tflops, double* reserved);

#ifdef __cplusplus
}
#endif
#endif /* HARD_B200_HARD_PROBE_H */

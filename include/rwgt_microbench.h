/* include/rwgt_microbench.h — measurement aid for the roofline of bench.py (MEASURED_PEAKS.json
 * has no FP64/FP32 FMA figure).  Lives in its own library, paper_2312_07440_b200/librwgt_microbench.so
 * (csrc/microbench.cu); it is not part of the reweighting ABI of include/rwgt.h and librwgt.so does not contain it. */
#ifndef RWGT_MICROBENCH_H
#define RWGT_MICROBENCH_H
#ifdef __cplusplus
extern "C" {
#endif

/* Runs a register-resident FMA chain on the CURRENT device and writes the sustained rate in TFLOP/s (2 flop per FMA,
 * best of 5 launches) to *out_tflops (HOST pointer).  Synchronises the device.  Returns 0, or -1 on a bad argument / CUDA error.
 * kind 0: FP64 FMA chain x = fma(x,a,b), 1: FP32 FMA chain, 2: FP64 tensor (mma m8n8k4) chain,
 * 3 / 4: FP64 FMA with three distinct register sources / with one source reused by consecutive FMAs (the operand
 * pattern of real complex arithmetic; register-file read bandwidth makes these slower than kind 0),
 * 5 / 6: the same two patterns in FP32, 7: FP64 FMA chains and DMMA chains concurrently on every SM, summed rate
 * (DFMA and DMMA share one pipe on B200: kind 7 = kind 0 = kind 2), 8 / 9 / 10: packed FP32 fma.rn.f32x2 (FFMA2) chains /
 * three distinct sources / one reused source (what the FP32 and mixed modes of librwgt.so issue). */
int rwgt_microbench_peak(int kind, double* out_tflops);

#ifdef __cplusplus
}
#endif
#endif /* RWGT_MICROBENCH_H */

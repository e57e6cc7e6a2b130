/*
 * xrdvi_measure.h -- microbenchmark of the SM pipes that bound the hot path.  NOT part of the product: it lives in its
 * own library, paper_2501_09308_b200/libxrdvi_measure.so (csrc/pipe_rates.cu; `python -m paper_2501_09308_b200.build
 * --measure`), which nothing in the product loads.  The constants of the ALU roofline in DESIGN.md ("Roofline") were
 * measured with it (profiles/r1_pipe_rates.md).
 */
#ifndef XRDVI_MEASURE_H
#define XRDVI_MEASURE_H

#ifdef __cplusplus
extern "C" {
#endif

/* Per-SM, per-clock rates of the pipes that bound the path.  rates float [9] (HOST): lane-operations per SM clock of
 * [0] FFMA, [1] FFMA2 (2 FMAs per lane), [2] MUFU.EX2, [3] MUFU.RCP, [4] the plain forward instruction mix (5 FP32 : 2
 * MUFU), [5] the plain backward mix (14 FP32 : 2 MUFU), [6] 7 FFMA2 : 2 MUFU, [7] EX2 and RCP chains run together
 * (MUFU operations per clock); [8] = SM clock (MHz) during the run.  Returns 0, or -6 on a CUDA error.        */
int xrdvi_pipe_rates(int device, float* rates);

#ifdef __cplusplus
}
#endif
#endif /* XRDVI_MEASURE_H */

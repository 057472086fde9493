/* tdprobe.h - C ABI of the bench-only probe library (libtdprobe.so).  Not part of the product: bench.py uses it to
 * measure, on the box it runs on, the arithmetic peaks its roofline fractions are quoted against (SURVEY.md 7.1 step 0,
 * 8(d)); libtdlike.so neither links nor calls it. */
#ifndef TDPROBE_H_
#define TDPROBE_H_

#ifdef __cplusplus
extern "C" {
#endif

/* td_probe_throughput - arithmetic throughput of `device` measured with register-resident dependent chains (no memory
 * traffic), 8 CTAs of 256 threads per SM:
 *   kind 0  DFMA chains (vector fp64 pipe),     kind 1  mma.sync.m8n8k4.f64 chains (fp64 tensor pipe),
 *   kind 2  both interleaved in the same warps,  kind 3  DADD chains (1 flop per instruction),
 *   kind 4  FFMA chains (fp32 pipe; the roofline of the fp32 evaluation mode).
 * tflops (HOST pointer) receives the best of 5 timed launches in TFLOP/s.  Synchronous; uses the legacy default stream.
 * Returns 0 on success, 1 for a bad argument, 4 for a CUDA failure (the td_status values of tdlike.h). */
int td_probe_throughput(int kind, int device, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* TDPROBE_H_ */

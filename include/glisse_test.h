/*
 * glisse_test.h — measurement and test hooks of libglisse.  NOT part of the library's interface
 * (include/glisse.h): bench.py uses them to count launches, time the dominant kernel and measure the
 * FP64 peak; the tests use them to evaluate device primitives one by one and to read the
 * Kepler-solver statistics.  Same conventions as glisse.h (0 / negative status, never throws).
 */
#ifndef GLISSE_TEST_H_
#define GLISSE_TEST_H_

#include "glisse.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernels the library has launched for this sim so far (bench.py's gpu_launches). */
long long glisse_launch_count(glisse_sim* sim);

/* Device time in milliseconds spent in particle kernels since the last call (or since create), and
 * the number of chunks' worth of launches it covers.  Measured with CUDA events recorded on the
 * sim's own stream around every run of back-to-back particle-kernel launches (the segment launches
 * of a chunk overlap each other by design, so they are timed together).  Synchronises. */
int glisse_particle_kernel_time(glisse_sim* sim, double* ms, long long* launches);

/*
 * Measure this GPU's plain FP64 FMA rate with a register-resident DFMA loop (no memory
 * traffic): returns the achieved FLOP/s (2 per DFMA) in *flops over a kernel of roughly
 * `millis` milliseconds on `device`, `stream` may be NULL.  Reported beside the nominal
 * roofline denominator of the ALU-bound particle kernel (MEASURED_PEAKS.json has no FP64 figure).
 */
int glisse_fp64_peak_probe(int device, void* stream, double millis, double* flops);

/*
 * Evaluate one device primitive of the CUDA path on an array, on device 0.
 * in/out are HOST or device arrays.  which = 0 rsqrt (in[n] -> out[n]), 1 reciprocal, 2 reciprocal
 * to 2^-39 (Newton updates only), 3 sin x - x and cos x - 1 (in[n] -> out[2n], interleaved),
 * 4 (5: with the third-order starting point, guess_order 3) one Kepler drift (step a5) per body: in[10n] = {mu, dt, kepler_iters, kepler_tol, x, y, z, vx,
 * vy, vz}, out[7n] = {flag, x, y, z, vx, vy, vz}; mu, kepler_iters and kepler_tol are taken from
 * body 0 for all bodies (constants of a run, warp-uniform in the kernel); dt is per body.  Synchronises.
 */
int glisse_test_primitive(int which, long long n, const double* in, double* out);

/*
 * Kepler-solver statistics (a warp runs as long as its slowest lane).  After
 * glisse_solver_stats_enable(sim, 1) the particle kernel runs an instrumented instantiation that
 * counts, per warp and per step, the fast-solver iterations the warp executed and whether it took the
 * definition's (slow) solver; glisse_solver_stats returns the totals since enable: warp_steps (warp
 * drift calls), warp_iters (fast-solver iterations summed over them), warp_slow (calls that entered
 * the slow path).  Synchronises.  Results of the integration are unchanged.
 */
int glisse_solver_stats_enable(glisse_sim* sim, int on);
int glisse_solver_stats(glisse_sim* sim, long long* warp_steps, long long* warp_iters, long long* warp_slow);

#ifdef __cplusplus
}
#endif
#endif /* GLISSE_TEST_H_ */

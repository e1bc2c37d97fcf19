/*
 * lh_diag.h -- diagnostics of liblh.so.  Not part of the method's boundary (include/lh.h): these calls serve
 * bench.py (roofline denominator, launch count), the CPU pins of the kernel's FP64 primitives, and the checking
 * build (liblh_check.so, -DLH_BOUNDS_CHECK) that tests/test_gpu_bounds.py drives.
 */
#ifndef LH_DIAG_H_
#define LH_DIAG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernels this host thread has launched through the library so far. */
long long lh_launch_count(void);

/* Diagnostic: runs a register-resident chain of dependent-free FP64 FMAs on every
 * SM for `iters` iterations and returns the achieved FP64 FLOP/s in *flops_per_s
 * (2 per FMA) and the kernel time in *seconds (CUDA events on the set stream;
 * synchronises).  Used by bench.py as the measured FP64 CUDA-core roofline. */
int lh_fp64_peak_probe(int iters, double *flops_per_s, double *seconds);

/* HOST evaluation of the kernel's own FP64 primitives (csrc/lh_math.cuh compiles for host and
 * device; on the host the 20-bit MUFU seeds are emulated by truncated exact quotients), so that
 * CPU-only tests can pin them against libm / arbitrary precision.  out[k] = fn(a[k], b[k]):
 *   fn 0  1/a            1  sqrt(a)        2  1/sqrt(a)
 *      3  atan(a/b), b > 0                 4  atanh(a/b), |a| < b, 1 - |a|/b > 2^-16
 *      5  1/a via the shared-seed pair (a, b)     6  1/a via the shared-seed quadruple (a, b, a+b, 2b)
 * No CUDA call is made.  LH_EINVAL for an unknown fn or a NULL pointer (b may be NULL for fn 0-2). */
int lh_math_host_eval(int fn, const double *a, const double *b, size_t n, double *out);

/* Hex SHA-256 of the sources and headers this library was compiled from (csrc/ files and include/ headers, in the
 * order paper_2004_06352_b200/_build.py lists them), or "unknown" when it was built by hand.  The libraries are
 * git-ignored and travel out of band, so a test that is about to vouch for the kernel with a prebuilt library
 * compares this with the hash of the tree it runs in (tests/bounds_child.py, tests/test_abi_cpu.py). */
const char *lh_source_hash(void);

#ifdef LH_BOUNDS_CHECK
/* Checking build only.  The address ranges superpose_kernel may touch on behalf of the caller: reset, add one range
 * [p, p + bytes) (LH_EINVAL when the list is full), and read the DEVICE counter of refused accesses (synchronises;
 * -1 on a CUDA error).  One host thread. */
int lh_debug_bounds_reset(void);
int lh_debug_bounds_add(const void *p, unsigned long long bytes);
long long lh_debug_violations(void);
#endif

#ifdef __cplusplus
}
#endif
#endif /* LH_DIAG_H_ */

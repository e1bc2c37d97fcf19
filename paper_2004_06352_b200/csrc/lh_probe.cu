// lh_probe.cu -- FP64 issue-cost microbenchmarks behind lh_fp64_issue_probe (include/lh.h).
//
// They measure what DESIGN.md sec. 7 builds on: how many dispatch cycles of an SM sub-partition
// one warp-wide FP64 instruction costs depending on where its operands come from, and what a
// non-FP64 instruction costs when it is mixed into a saturated FP64 stream.  One group =
// 12 independent FP64 instructions (+ `extra` other instructions); every thread runs `iters`
// groups; the result is cycles per group per sub-partition at the device's SM clock.
#include <cuda_runtime.h>

#include "lh_kernels.h"

namespace lh {

constexpr int NCH = 12;
struct ProbeTable {
    double v[64];
};

template <int V, int EXTRA>
__global__ void __launch_bounds__(128) issue_probe_kernel(int iters, double seed, double *sink, const __grid_constant__ ProbeTable tab) {
    __shared__ double sm[64];
    if (threadIdx.x < 64) sm[threadIdx.x] = tab.v[threadIdx.x];
    __syncthreads();
    double a[NCH], b[NCH], c[NCH];
    int x[8];
    float f[8];
#pragma unroll
    for (int i = 0; i < NCH; ++i) {
        a[i] = seed + i + threadIdx.x * 1e-9;
        b[i] = 1.0 - 1e-12 * (i + 1) - threadIdx.x * 1e-15;
        c[i] = 1e-12 * (i + 1) + threadIdx.x * 1e-17;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        x[i] = threadIdx.x * 7 + i;
        f[i] = 1.0f + i + threadIdx.x;
    }
    for (int it = 0; it < iters; ++it) {
        const int j = (it * 4) & 31;  // warp-uniform index into the parameter table
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
            if (V == 0) a[i] = fma(a[i], 1.0 - 1e-12, 1e-12);   // immediates / uniform constants
            if (V == 1) a[i] = fma(b[i], c[i], a[i]);           // three distinct vector registers
            if (V == 2) a[i] = fma(a[i], b[i], a[i]);           // two distinct (one repeated)
            if (V == 3) a[i] = a[i] * b[i];                     // DMUL, two registers
            if (V == 4) a[i] = fma(a[i], tab.v[j + (i & 3)], c[i]);  // one uniform operand (LDCU from the parameters)
            if (V == 5) a[i] = fma(a[i], b[0], c[i]);           // one register shared by consecutive instructions (.reuse)
        }
#pragma unroll
        for (int e = 0; e < EXTRA; ++e) {
            if (V == 10) asm volatile("lop3.b32 %0, %0, %1, 0x5555, 0x96;" : "+r"(x[e % 8]) : "r"(x[(e + 1) % 8]));
            if (V == 11) asm volatile("fma.rn.f32 %0, %0, %1, %0;" : "+f"(f[e % 8]) : "f"(f[(e + 3) % 8]));
            if (V == 12) { double y; asm volatile("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a[e % NCH])); b[(e + 5) % NCH] = y; }
            if (V == 13) b[e % NCH] = sm[(it + e) & 63];
        }
        if (V >= 10) {
#pragma unroll
            for (int i = 0; i < NCH; ++i) a[i] = a[i] * b[i];
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < NCH; ++i) s += a[i] + b[i] + c[i];
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i] + f[i];
    if (s == 123.456) sink[0] = s;  // never true; keeps everything alive
}

template <int V, int EXTRA>
static cudaError_t go(int iters, int blocks, double *sink, cudaStream_t st) {
    ProbeTable t;
    for (int i = 0; i < 64; ++i) t.v[i] = 1.0 - 1e-13 * i;
    issue_probe_kernel<V, EXTRA><<<blocks, 128, 0, st>>>(iters, 1.0, sink, t);
    return cudaGetLastError();
}

// variant: 0-5 operand patterns of the FP64 instruction; 10-13 a DMUL stream plus `extra`
// (0, 2, 4 or 8) LOP3 / FFMA / MUFU.RCP64H(+MOV) / LDS per group.
cudaError_t launch_issue_probe(int variant, int extra, int iters, int blocks, double *sink, cudaStream_t st) {
    switch (variant) {
        case 0: return go<0, 0>(iters, blocks, sink, st);
        case 1: return go<1, 0>(iters, blocks, sink, st);
        case 2: return go<2, 0>(iters, blocks, sink, st);
        case 3: return go<3, 0>(iters, blocks, sink, st);
        case 4: return go<4, 0>(iters, blocks, sink, st);
        case 5: return go<5, 0>(iters, blocks, sink, st);
        default: break;
    }
#define LH_EXTRA(V)                                                  \
    case V:                                                          \
        if (extra == 0) return go<V, 0>(iters, blocks, sink, st);    \
        if (extra == 2) return go<V, 2>(iters, blocks, sink, st);    \
        if (extra == 4) return go<V, 4>(iters, blocks, sink, st);    \
        if (extra == 8) return go<V, 8>(iters, blocks, sink, st);    \
        return cudaErrorInvalidValue;
    switch (variant) {
        LH_EXTRA(10)
        LH_EXTRA(11)
        LH_EXTRA(12)
        LH_EXTRA(13)
        default: return cudaErrorInvalidValue;
    }
#undef LH_EXTRA
}

}  // namespace lh

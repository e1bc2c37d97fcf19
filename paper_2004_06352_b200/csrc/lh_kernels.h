// lh_kernels.h -- launch interface between the C ABI (lh_api.cu) and the kernels.
#pragma once
#include <cuda_runtime.h>

#include "lh_math.cuh"
#include "lh_pack.h"

namespace lh {

struct EvalParams {
    const LensK *table;         // [nmodel][nlens], each model sorted by class
    const ModelRanges *ranges;  // [nmodel]
    const MathTables *math;     // device copy of the atan / atanh reduction tables
    int nlens, nmodel;
    int any_extreme;            // some model holds CLS_EXTREME lenses (selects the kernel instantiation)
    double x0, y0, dx;
    int nx, ny;
    long long plane;  // nx*ny
    double *out[9];   // ax ay a11 a12 a22 kappa gamma1 gamma2 mu; nullptr = not wanted
    int tiles_x, tiles_y;  // filled by launch_eval
};

cudaError_t launch_eval(const EvalParams &P, cudaStream_t stream);
cudaError_t launch_dfma_probe(int iters, int blocks, double *sink, cudaStream_t stream);

}  // namespace lh

// lh_kernels.h -- launch interface between the C ABI (lh_api.cu) and the kernels.
#pragma once
#include <cuda_runtime.h>

#include "lh_math.cuh"
#include "lh_pack.h"

namespace lh {

// Records one launch carries in its kernel parameters (constant bank 0, 32 764 bytes at most):
// 160 x 192 B of lens constants + 160 x 8 B of class boundaries + a header of about 250 bytes.
constexpr int LAUNCH_RECORDS = 160;
constexpr int LAUNCH_MODELS = 160;  // models that may share one launch (blockIdx.y)
constexpr int DBG_RANGES = 16;      // checking build (-DLH_BOUNDS_CHECK): address ranges a launch may touch

struct LaunchParams {
    double x0, y0, dx;
    Consts kc;               // 1/3, 1/5, 3/8 as launch-parameter VALUES (lh_math.cuh: kept in registers, not rematerialised)
    long long plane;         // nx*ny
    double *out[9];          // ax ay a11 a12 a22 kappa gamma1 gamma2 mu; nullptr = not wanted; [nmodel][ny][nx]
    double *carry;           // [5][ny][nx] accumulators handed from one lens chunk of a model to the next
    const MathTables *math;  // device copy of the atan / atanh reduction tables
    int nx, ny, tiles_x;     // ny = rows of THIS launch (a row slab of the grid when j0 > 0)
    int j0;                  // first grid row of the slab: pixel row j of the launch sits at y0 + (j0 + j) dx
    int model0;              // global index of the launch's first model (blockIdx.y = model - model0)
    int stride;              // records per model in table[]
    int first, last;         // this launch holds the first / last lens chunk of its model(s)
    int stats_n;             // stats only: models folded into out[] / m2[] including this launch's
    int stats;               // 0: out[] are per-model planes.  1 / 2: out[] are running MEANS over models and m2[] the
                             // running sums of squared deviations (Welford); 2 = last model: m2[] is divided by the count
    double *m2[9];           // stats only; nullptr = variance of that plane not wanted
    const double *px, *py;   // POINTS variants only: coordinates of "pixel" i (then ny = 1, nx = number of points)
#ifdef LH_BOUNDS_CHECK
    const char *dbg_lo[DBG_RANGES], *dbg_hi[DBG_RANGES];  // checking build: the address ranges this launch may touch
    unsigned long long *dbg_count;                        // DEVICE counter of refused accesses
    int dbg_n;
#endif
    unsigned short cls_end[LAUNCH_MODELS][CLS_COUNT];  // per model: end of each class, relative to its slice
    LensK table[LAUNCH_RECORDS];
};
static_assert(sizeof(LaunchParams) <= 32764, "kernel parameter space");

// One call of the C ABI: nmodel packed tables (host memory) on one grid.
struct EvalJob {
    const LensK *table;         // HOST [nmodel][nlens], each model sorted by class
    const ModelRanges *ranges;  // HOST [nmodel]
    const MathTables *math;     // DEVICE
    int nlens, nmodel;
    // f4: lenses common to every model of the batch, evaluated ONCE into `carry`; every model then starts from
    // those accumulators (nullptr / 0 = none).  Needs nlens <= LAUNCH_RECORDS and carry != nullptr.
    const LensK *shared_table;  // HOST [nshared], sorted by class
    ModelRanges shared_ranges;
    int nshared;
    double x0, y0, dx;
    int nx, ny;      // ny = rows evaluated by this job
    int j0;          // first grid row (row slab of a larger grid; out[] / carry already point at that row)
    long long plane; // doubles between consecutive models / accumulators (the FULL plane, >= nx*ny)
    const double *px, *py;  // DEVICE, both or neither: evaluate at these nx points (ny = 1) instead of the grid
    double *out[9];  // DEVICE
    double *m2[9];   // DEVICE, stats only (else all nullptr)
    int stats;       // 0 = per-model planes [nmodel][ny][nx]; 1 = mean / variance over the models, planes [ny][nx]
    double *carry;   // DEVICE, 5*nx*ny doubles; needed only when nlens > LAUNCH_RECORDS
    // optional second chain for batches of chunked models (all four or none): every other model runs on `aux` with
    // `carry2`; launch_eval forks `aux` from the job's stream (ev_fork) and joins it back (ev_join) before returning
    double *carry2 = nullptr;
    cudaStream_t aux = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    double *stats_scratch = nullptr;  // stats + two chains: DEVICE, 18 planes (mean, m2 of the odd-model chain)
#ifdef LH_BOUNDS_CHECK
    const char *dbg_lo[DBG_RANGES], *dbg_hi[DBG_RANGES];
    unsigned long long *dbg_count = nullptr;
    int dbg_n = 0;
#endif
};

// Enqueues every launch of the job on `stream`; adds the number of kernels launched to *launches.
cudaError_t launch_eval(const EvalJob &J, cudaStream_t stream, long long *launches);
cudaError_t launch_dfma_probe(int iters, int blocks, double *sink, cudaStream_t stream);

// lh_delens.cu (NEXT row f1)
cudaError_t launch_source_plane(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                                double *bx, double *by, int sms, cudaStream_t st);

}  // namespace lh

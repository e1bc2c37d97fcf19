// lh_noalloc.cu -- lh_grid_eval_noalloc (include/lh.h): the row-slab evaluation for callers that must not
// allocate device memory.
//
// Why it exists.  Every other entry point obtains two things from cudaMalloc the first time it needs them: the
// read-only atan / atanh reduction tables, and -- for a lens list longer than one launch can carry
// (lh::LAUNCH_RECORDS = 160) -- the `carry` planes through which one launch hands its five partial sums per pixel
// to the next.  Some programs cannot let a library do that:
//   - the process runs under a memory manager that has taken the whole device (a framework's caching allocator, a
//     batch system that gives each job a fixed partition): a cudaMalloc made behind its back fails, or succeeds
//     and breaks the manager's accounting;
//   - the call sits in a loop that must not stall (a sampler step, a service with a latency budget): cudaMalloc
//     and cudaFree synchronise the device, so one of them in the middle of the loop stops every stream;
//   - the deployment rules say "all device memory is reserved at start-up, none afterwards".
// For them the two buffers live here as file-scope `static __device__` arrays.  The loader reserves them on every
// GPU that loads liblh.so, for the life of the process: NOALLOC_CARRY_BYTES (40 MiB) + sizeof(MathTables)
// (32 KB).  The price is a fixed maximum job size, LH_NOALLOC_MAX_PIXELS per call (a larger grid is covered
// by several calls, one row slab each), and one buffer shared by all calls.
//
// The kernel is the library's superpose_kernel, unchanged; this file only decides where its `carry` and `math`
// pointers point.  In HOST code the name of a __device__ array is a host-side shadow symbol, not a device
// address, so device_buffers() asks cudaGetSymbolAddress once per device and the launches are given that answer.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/lh.h"
#include "lh_kernels.h"

namespace lh {  // lh_api.cu: this host thread's stream, error text and launch counter
cudaStream_t api_stream();
int api_fail(int code, const char *msg);
void api_clear_error();
long long *api_launch_counter();
}  // namespace lh

namespace {

constexpr long long MAX_PIXELS = LH_NOALLOC_MAX_PIXELS;
constexpr size_t NOALLOC_CARRY_BYTES = (size_t)5 * MAX_PIXELS * sizeof(double);
static_assert(NOALLOC_CARRY_BYTES == (size_t)40 << 20, "lh.h states 40 MiB");

int fail(int code, const char *fmt, ...) {
    char msg[384];
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(msg, sizeof(msg), fmt, ap);
    va_end(ap);
    return lh::api_fail(code, msg);
}

#ifndef LH_BOUNDS_CHECK  // the checking build closes this entry point (below) and reserves nothing
constexpr int MAX_LENSES = LH_NOALLOC_MAX_LENSES;
constexpr int MAX_DEVICES = 64;

// ---- the scratch itself: device memory that belongs to the library image, not to any allocator ----------------
// five accumulator planes (alpha_x, alpha_y and the three Hessian sums) of up to MAX_PIXELS pixels each
static __device__ __align__(256) double g_carry[5 * MAX_PIXELS];
// the reduction tables of lh_math.cuh, uploaded by the first call on each device
static __device__ __align__(256) lh::MathTables g_math;

// host side: everything below is guarded by g_mu, one caller at a time
std::mutex g_mu;
lh::LensK g_table[MAX_LENSES];  // packed lens records of the call in progress (copied into the launch parameters
lh::ModelRanges g_ranges;       // by launch_eval, so the next call may overwrite them)
lh::MathTables g_host_math;
bool g_host_math_ready = false;
struct PerDevice {
    double *carry = nullptr;          // DEVICE address of g_carry on that device
    const lh::MathTables *math = nullptr;  // DEVICE address of g_math on that device
    bool ready = false;
} g_dev[MAX_DEVICES];


// Set-up of the current device, on the first call that reaches it: look up where g_carry and g_math live on THIS
// device (each device that loaded the library has its own copy at its own address) and fill the tables.  The
// upload is a plain synchronous cudaMemcpy.  Returns LH_OK or LH_ECUDA.
int device_buffers(int dev, PerDevice **out) {
    PerDevice &D = g_dev[dev];
    if (!D.ready) {
        void *pc = nullptr, *pm = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&pc, g_carry);
        if (e != cudaSuccess) return fail(LH_ECUDA, "lh_grid_eval_noalloc: cudaGetSymbolAddress(carry): %s", cudaGetErrorString(e));
        e = cudaGetSymbolAddress(&pm, g_math);
        if (e != cudaSuccess) return fail(LH_ECUDA, "lh_grid_eval_noalloc: cudaGetSymbolAddress(tables): %s", cudaGetErrorString(e));
        if (!g_host_math_ready) {
            lh::fill_math_tables(g_host_math);
            g_host_math_ready = true;
        }
        e = cudaMemcpy(pm, &g_host_math, sizeof(g_host_math), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return fail(LH_ECUDA, "lh_grid_eval_noalloc: table upload: %s", cudaGetErrorString(e));
        D.carry = static_cast<double *>(pc);
        D.math = static_cast<const lh::MathTables *>(pm);
        D.ready = true;
    }
    *out = &D;
    return LH_OK;
}

const char *PLANE_NAMES[9] = {"ax", "ay", "a11", "a12", "a22", "kappa", "gamma1", "gamma2", "mu"};

int check_output(const double *p, const char *name) {
    if ((reinterpret_cast<uintptr_t>(p) & 7u) != 0) return fail(LH_EINVAL, "output %s is not 8-byte aligned", name);
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return fail(LH_EINVAL, "output %s is not a device pointer", name);
    }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(LH_EINVAL, "output %s is not a device pointer", name);
    return LH_OK;
}
#endif  // !LH_BOUNDS_CHECK

}  // namespace

extern "C" int lh_grid_eval_noalloc(const lh_lens *lenses, int nlens, const lh_grid *g, int j0, int nrows,
                                    const lh_outputs *o) {
    lh::api_clear_error();
#ifdef LH_BOUNDS_CHECK
    // the checking build (liblh_check.so) registers address ranges per launch through lh_api.cu; this entry point
    // is not wired into that and is closed there rather than run unchecked
    (void)lenses; (void)nlens; (void)g; (void)j0; (void)nrows; (void)o;
    return fail(LH_EINVAL, "lh_grid_eval_noalloc is not part of the checking build");
#else
    // ---- arguments: everything is checked before the first CUDA call that could enqueue work
    if (nlens < 0) return fail(LH_EINVAL, "nlens must be >= 0");
    if (nlens > 0 && !lenses) return fail(LH_EINVAL, "lenses is NULL");
    if (nlens > MAX_LENSES)
        return fail(LH_EINVAL, "lh_grid_eval_noalloc: %lld lenses, the fixed host table holds LH_NOALLOC_MAX_LENSES = %d",
                    (long long)nlens, MAX_LENSES);
    if (!g) return fail(LH_EINVAL, "grid is NULL");
    if (g->nx <= 0 || g->ny <= 0) return fail(LH_EINVAL, "grid: nx and ny must be > 0");
    if (!(std::isfinite(g->x0) && std::isfinite(g->y0) && std::isfinite(g->dx)) || !(g->dx > 0.0))
        return fail(LH_EINVAL, "grid: x0, y0 must be finite and dx > 0");
    if (j0 < 0 || nrows < 1 || (long long)j0 + nrows > g->ny) return fail(LH_EINVAL, "row slab outside the grid");
    const long long npix = (long long)g->nx * nrows;
    if (npix > MAX_PIXELS)
        return fail(LH_EINVAL,
                    "lh_grid_eval_noalloc: slab of %lld pixels, the static scratch holds LH_NOALLOC_MAX_PIXELS = %lld "
                    "(cover the grid with several calls of fewer rows)", npix, (long long)MAX_PIXELS);
    if (!o) return fail(LH_EINVAL, "outputs is NULL");
    double *p[9] = {o->ax, o->ay, o->a11, o->a12, o->a22, o->kappa, o->gamma1, o->gamma2, o->mu};
    bool any = false;
    for (int k = 0; k < 9; ++k) {
        if (!p[k]) continue;
        any = true;
        int rc = check_output(p[k], PLANE_NAMES[k]);
        if (rc) return rc;
    }
    if (!any) return fail(LH_EINVAL, "no output plane requested");

    std::lock_guard<std::mutex> lock(g_mu);
    // step a1 into the fixed host table (validates every lens; nothing has been enqueued yet)
    char msg[384];
    if (lh::pack_model(lenses, nlens, g_table, &g_ranges, msg, sizeof(msg), 0) != 0) return lh::api_fail(LH_EINVAL, msg);

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(LH_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(LH_ECUDA, "device index %d outside [0, %d)", dev, MAX_DEVICES);
    PerDevice *D = nullptr;
    int rc = device_buffers(dev, &D);
    if (rc) return rc;

    // One model, one launch chain on the caller's stream: no second stream, no events.  The slab is presented as
    // lh_grid_eval_rows presents it -- planes of nrows x nx whose row 0 is grid row j0 -- and the carry planes
    // are laid out the same way at the start of g_carry (plane stride = the slab's pixel count).
    lh::EvalJob J = {};
    J.table = g_table;
    J.ranges = &g_ranges;
    J.math = D->math;
    J.nlens = nlens;
    J.nmodel = 1;
    J.shared_table = nullptr;
    J.nshared = 0;
    J.x0 = g->x0; J.y0 = g->y0; J.dx = g->dx;
    J.nx = g->nx; J.ny = nrows;
    J.j0 = j0;
    J.plane = npix;
    J.px = nullptr; J.py = nullptr;
    for (int k = 0; k < 9; ++k) { J.out[k] = p[k]; J.m2[k] = nullptr; }
    J.stats = 0;
    J.carry = D->carry;
    e = lh::launch_eval(J, lh::api_stream(), lh::api_launch_counter());
    if (e != cudaSuccess) return fail(LH_ECUDA, "lh_grid_eval_noalloc: launch: %s", cudaGetErrorString(e));
    return LH_OK;
#endif
}

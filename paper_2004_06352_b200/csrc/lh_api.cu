// lh_api.cu -- the C ABI of liblh.so (include/lh.h): argument checks, host packing,
// staging of the packed table, launch.  No arithmetic of the method lives here.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <thread>
#include <new>
#include <vector>

#include "../../include/lh.h"
#include "../../include/lh_diag.h"
#include "lh_kernels.h"

namespace lh {
cudaError_t launch_delens(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                          const double *sources, int ns, lh_image *images, long long max_images,
                          unsigned long long *count, int sms, cudaStream_t st, long long *launches);
cudaError_t launch_delens_dev(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                              const double *dsources, int ns, lh_image *images, long long max_images,
                              unsigned long long *count, int sms, cudaStream_t st, long long *launches);
cudaError_t launch_constraint_points(const lh_constraint *c, int K, double *cx, double *cy, cudaStream_t st);
cudaError_t launch_barycentre(const lh_constraint *c, int K, const double *ax, const double *ay, int nsources, double *src,
                              cudaStream_t st);
cudaError_t launch_assign_and_sum(const lh_constraint *c, int K, const lh_image *im, const unsigned long long *count,
                                  long long cap, double *pred, double *term, double *chi2, long long *nimages,
                                  cudaStream_t st);
}

namespace {

using lh::LensK;
using lh::ModelRanges;

// Per-host-thread state: stream, last error, the host buffer the lens tables are packed
// into, and two cached device buffers.  The packed records travel to the device inside the
// kernel parameters (lh_kernels.h), copied by the launch itself, so the host buffer may be
// rewritten as soon as launch_eval returns.  `d_carry` (accumulators handed from one lens
// chunk of a model to the next) is reused across calls: stream order protects it on one
// stream, ev_done + cudaStreamWaitEvent across a stream change.
// Everything that lives on ONE device: cached buffers, events, the copy stream.  A host thread may switch
// devices between calls (cudaSetDevice / torch.cuda.set_device); each device then gets its own state.
struct DeviceState {
    double *d_carry = nullptr;
    size_t carry_bytes = 0;
    cudaEvent_t ev_done = nullptr;
    cudaStream_t last_stream = nullptr;
    bool busy = false;

    double *d_planes = nullptr;  // cached device planes for the *_host entry point
    size_t planes_bytes = 0;
    static const int PIECES = 8;  // pipeline depth of the *_host entry point (compute piece k+1 | copy piece k)
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_piece[PIECES] = {};
    cudaEvent_t ev_copied[PIECES] = {};  // piece k has landed in the pinned ring (pageable host planes only)
    char *h_ring = nullptr;              // pinned bounce ring of the *_host entry points: 2 slots
    size_t ring_bytes = 0;
    double *d_sink = nullptr;
    char *d_chi = nullptr;  // scratch of lh_chi2 (deflection planes, constraint arrays, sources, images)
    size_t chi_bytes = 0;
    cudaEvent_t ev_chi = nullptr;  // end of the last lh_chi2 that used d_chi, on chi_stream (same protocol as d_carry)
    cudaStream_t chi_stream = nullptr;
    bool chi_busy = false;
    cudaStream_t aux_stream = nullptr;  // second launch chain of batches of chunked models (lh_kernels.cu)
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t piece_stream = nullptr;  // the odd pieces of the *_host entry points (one map): their launch tails overlap
    cudaEvent_t ev_pfork = nullptr, ev_pjoin = nullptr;
};

struct Context {
    cudaStream_t stream = nullptr;
    char err[512] = {0};
    long long launches = 0;

    std::vector<LensK> h_table, h_shared;
    std::vector<ModelRanges> h_ranges;

    static const int MAX_DEVICES = 64;
    DeviceState dev[MAX_DEVICES];

    ~Context() {
        // process teardown: the CUDA runtime may already be gone; leak deliberately.
    }
};

thread_local Context ctx;

#ifdef LH_BOUNDS_CHECK
// Checking build only (liblh_check.so): the address ranges the caller allows superpose_kernel to touch
// (lh_debug_bounds_add) and the device counter of refused accesses.  Test infrastructure: one host thread.
struct DebugBounds {
    const char *lo[lh::DBG_RANGES], *hi[lh::DBG_RANGES];
    int n = 0;
    unsigned long long *d_count = nullptr;
} dbg;
#endif

// state of the device that is current on this host thread
DeviceState &DS() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= Context::MAX_DEVICES) d = 0;
    return ctx.dev[d];
}

// The atan / atanh reduction tables (lh_math.cuh): one read-only device copy per device,
// made on first use and kept for the life of the process.
const lh::MathTables *device_math_tables(int dev, cudaError_t *err) {
    static std::mutex mu;
    static const lh::MathTables *cache[64] = {nullptr};
    std::lock_guard<std::mutex> lock(mu);
    *err = cudaSuccess;
    if (dev < 0 || dev >= 64) { *err = cudaErrorInvalidDevice; return nullptr; }
    if (!cache[dev]) {
        static lh::MathTables host;
        lh::fill_math_tables(host);
        void *d = nullptr;
        if ((*err = cudaMalloc(&d, sizeof(host))) != cudaSuccess) return nullptr;
        if ((*err = cudaMemcpy(d, &host, sizeof(host), cudaMemcpyHostToDevice)) != cudaSuccess) { cudaFree(d); return nullptr; }
        cache[dev] = static_cast<const lh::MathTables *>(d);
    }
    return cache[dev];
}

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(ctx.err, sizeof(ctx.err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) return fail(LH_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));     \
    } while (0)

const int NPLANES = 9;

void planes_of(const lh_outputs *o, double *p[NPLANES]) {
    p[0] = o->ax; p[1] = o->ay; p[2] = o->a11; p[3] = o->a12; p[4] = o->a22;
    p[5] = o->kappa; p[6] = o->gamma1; p[7] = o->gamma2; p[8] = o->mu;
}

int check_grid(const lh_grid *g, int nmodel) {
    if (!g) return fail(LH_EINVAL, "grid is NULL");
    if (g->nx <= 0 || g->ny <= 0) return fail(LH_EINVAL, "grid: nx and ny must be > 0");
    if (!(std::isfinite(g->x0) && std::isfinite(g->y0) && std::isfinite(g->dx)) || !(g->dx > 0.0))
        return fail(LH_EINVAL, "grid: x0, y0 must be finite and dx > 0");
    const long double tot = (long double)g->nx * g->ny * nmodel;
    if (tot >= (long double)(1ULL << 40)) return fail(LH_EINVAL, "grid: nmodel*nx*ny must be < 2^40");
    return LH_OK;
}

int check_device_ptr(const double *p, const char *name) {
    if ((reinterpret_cast<uintptr_t>(p) & 7u) != 0) return fail(LH_EINVAL, "output %s is not 8-byte aligned", name);
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(LH_EINVAL, "output %s is not a device pointer", name);
    }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(LH_EINVAL, "output %s is not a device pointer", name);
    return LH_OK;
}

const char *PLANE_NAMES[NPLANES] = {"ax", "ay", "a11", "a12", "a22", "kappa", "gamma1", "gamma2", "mu"};

// Validate + pack + launch.  `dev_out` are device planes (already checked).
// Optional parts of a job.
struct EvalOpts {
    double **m2 = nullptr;            // != nullptr selects the statistics mode: dev_out are mean planes, m2 variance planes
    const lh_lens *shared = nullptr;  // lenses common to every model (f4), evaluated once
    int nshared = 0;
    int j0 = 0, nrows = -1;           // rows [j0, j0 + nrows) of the grid only (dev_out point at row j0); default all
    int buf_row0 = 0;                 // row, inside planes of g->ny rows, at which dev_out point (carry is laid out alike)
    const double *px = nullptr, *py = nullptr;  // DEVICE: evaluate at these g->nx points instead of a grid (g->ny = 1)
    // >= 0: the models were validated and packed into ctx.h_table / ctx.h_ranges by pack_all() already and this job
    // evaluates `nmodel` of them starting at model `packed0` (`lenses` is then not read)
    int packed0 = -1;
    // the caller has already made the carry buffer safe for this job and will record its end of use itself (the pieces
    // of eval_host alternate between two streams and touch disjoint rows of one carry buffer)
    bool carry_guard_by_caller = false;
    cudaStream_t stream_override = nullptr;  // != nullptr: enqueue on this stream instead of the thread's
};

// a1 for a whole call: validate + pack nmodel x nlens lenses into ctx.h_table / ctx.h_ranges.  Nothing is enqueued.
int pack_all(const lh_lens *lenses, int nmodel, int nlens) {
    try {
        ctx.h_table.resize((size_t)nmodel * (size_t)nlens);
        ctx.h_ranges.resize((size_t)nmodel);
    } catch (const std::bad_alloc &) {
        return fail(LH_EINVAL, "out of host memory packing %d x %d lenses", nmodel, nlens);
    }
    for (int m = 0; m < nmodel; ++m) {
        if (lh::pack_model(lenses + (size_t)m * nlens, nlens, ctx.h_table.data() + (size_t)m * nlens,
                           ctx.h_ranges.data() + m, ctx.err, sizeof(ctx.err), m) != 0)
            return LH_EINVAL;  // message already written
    }
    return LH_OK;
}

// The carry buffer of this device: at least `need` bytes, safe to use on stream `s` once this returns.
int ensure_carry(size_t need, cudaStream_t s) {
    if (!DS().ev_done) CU(cudaEventCreateWithFlags(&DS().ev_done, cudaEventDisableTiming));
    if (need > DS().carry_bytes) {
        if (DS().busy) CU(cudaEventSynchronize(DS().ev_done));  // the old buffer is no longer in use
        if (DS().d_carry) cudaFree(DS().d_carry);
        DS().d_carry = nullptr;
        DS().carry_bytes = 0;
        CU(cudaMalloc(&DS().d_carry, need));
        DS().carry_bytes = need;
    }
    if (need && DS().busy && DS().last_stream != s) CU(cudaStreamWaitEvent(s, DS().ev_done, 0));
    return LH_OK;
}

// The second launch chain of chunked models (lh_kernels.cu): its stream and the fork / join events, made once per device.
int ensure_aux_stream() {
    if (!DS().aux_stream) CU(cudaStreamCreateWithFlags(&DS().aux_stream, cudaStreamNonBlocking));
    if (!DS().ev_fork) CU(cudaEventCreateWithFlags(&DS().ev_fork, cudaEventDisableTiming));
    if (!DS().ev_join) CU(cudaEventCreateWithFlags(&DS().ev_join, cudaEventDisableTiming));
    return LH_OK;
}

int eval_device(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, double *dev_out[NPLANES],
                const EvalOpts &opt = EvalOpts()) {
    double **dev_m2 = opt.m2;
    const lh_lens *shared = opt.shared;
    const int nshared = opt.nshared, j0 = opt.j0;
    int nrows = opt.nrows;
    if (nrows < 0) nrows = g->ny;
    // a1: pack on the host (validates; nothing is enqueued if any lens is rejected)
    const int m_first = opt.packed0 >= 0 ? opt.packed0 : 0;
    if (opt.packed0 < 0) {
        int rc = pack_all(lenses, nmodel, nlens);
        if (rc) return rc;
    }

    lh::ModelRanges shared_ranges = {};
    if (nshared > 0) {
        try {
            ctx.h_shared.resize((size_t)nshared);
        } catch (const std::bad_alloc &) {
            return fail(LH_EINVAL, "out of host memory packing %d shared lenses", nshared);
        }
        if (lh::pack_model(shared, nshared, ctx.h_shared.data(), &shared_ranges, ctx.err, sizeof(ctx.err), -1) != 0)
            return LH_EINVAL;
    }

    cudaStream_t s = opt.stream_override ? opt.stream_override : ctx.stream;
    const size_t carry_one =
        (nlens > lh::LAUNCH_RECORDS || nshared > 0) ? (size_t)5 * g->nx * g->ny * sizeof(double) : 0;
    // batches of chunked models run as two interleaved launch chains, each with a carry buffer of its own
    // (statistics: the odd-model chain folds into scratch planes kept behind the two carry buffers)
    const bool two_chains = nlens > lh::LAUNCH_RECORDS && nmodel > 1 && nshared == 0;
    const size_t stats_scratch = (two_chains && dev_m2) ? (size_t)18 * g->nx * g->ny * sizeof(double) : 0;
    const size_t carry_need = carry_one * (two_chains ? 2 : 1) + stats_scratch;
    // one chunked model on a grid: its two row halves run as two chains (lh_kernels.cu); not for the pieces of eval_host,
    // which are two chains themselves
    const bool row_halves = nlens > lh::LAUNCH_RECORDS && nmodel == 1 && !dev_m2 && nshared == 0 && !opt.px &&
                            !opt.carry_guard_by_caller;
    if (two_chains || row_halves) {
        int rc = ensure_aux_stream();
        if (rc) return rc;
    }
    if (!opt.carry_guard_by_caller) {
        int rc = ensure_carry(carry_need, s);
        if (rc) return rc;
    }

    int dev = 0;
    CU(cudaGetDevice(&dev));
    cudaError_t terr;
    lh::EvalJob J;
    J.math = device_math_tables(dev, &terr);
    if (!J.math) return fail(LH_ECUDA, "math tables: %s", cudaGetErrorString(terr));
    J.table = ctx.h_table.data() + (size_t)m_first * nlens;
    J.ranges = ctx.h_ranges.data() + m_first;
    J.nlens = nlens;
    J.nmodel = nmodel;
    J.shared_table = nshared > 0 ? ctx.h_shared.data() : nullptr;
    J.shared_ranges = shared_ranges;
    J.nshared = nshared;
    J.x0 = g->x0; J.y0 = g->y0; J.dx = g->dx;
    J.nx = g->nx; J.ny = nrows;
    J.j0 = j0;
    J.plane = (long long)g->nx * g->ny;
    J.px = opt.px; J.py = opt.py;
    for (int k = 0; k < NPLANES; ++k) {
        J.out[k] = dev_out[k];
        J.m2[k] = dev_m2 ? dev_m2[k] : nullptr;
    }
    J.stats = dev_m2 ? 1 : 0;
    // carry is laid out like the planes it serves (g->ny rows of g->nx): a piece that starts at row buf_row0 of
    // those planes uses the same rows of the carry buffer
    J.carry = DS().d_carry ? DS().d_carry + (size_t)opt.buf_row0 * g->nx : nullptr;
    if (row_halves) {
        J.aux = DS().aux_stream;
        J.ev_fork = DS().ev_fork;
        J.ev_join = DS().ev_join;
    }
    if (two_chains) {
        J.carry2 = DS().d_carry + carry_one / sizeof(double);
        J.aux = DS().aux_stream;
        J.ev_fork = DS().ev_fork;
        J.ev_join = DS().ev_join;
        if (stats_scratch) J.stats_scratch = DS().d_carry + 2 * (carry_one / sizeof(double));
    }
#ifdef LH_BOUNDS_CHECK
    if (!dbg.d_count) {
        CU(cudaMalloc(&dbg.d_count, sizeof(unsigned long long)));
        CU(cudaMemset(dbg.d_count, 0, sizeof(unsigned long long)));
    }
    J.dbg_count = dbg.d_count;
    J.dbg_n = 0;
    for (int r = 0; r < dbg.n; ++r) { J.dbg_lo[J.dbg_n] = dbg.lo[r]; J.dbg_hi[J.dbg_n] = dbg.hi[r]; ++J.dbg_n; }
    // the library's own buffers: the carry / statistics scratch exactly as large as THIS job needs it (the cached
    // allocation may be larger), and the reduction tables
    if (carry_need) {
        J.dbg_lo[J.dbg_n] = reinterpret_cast<const char *>(DS().d_carry);
        J.dbg_hi[J.dbg_n] = reinterpret_cast<const char *>(DS().d_carry) + carry_need;
        ++J.dbg_n;
    }
    J.dbg_lo[J.dbg_n] = reinterpret_cast<const char *>(J.math);
    J.dbg_hi[J.dbg_n] = reinterpret_cast<const char *>(J.math) + sizeof(lh::MathTables);
    ++J.dbg_n;
#endif
    CU(lh::launch_eval(J, s, &ctx.launches));
    if (carry_need && !opt.carry_guard_by_caller) {
        CU(cudaEventRecord(DS().ev_done, s));
        DS().busy = true;
        DS().last_stream = s;
    }
    return LH_OK;
}

int check_common(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g) {
    if (nmodel < 1) return fail(LH_EINVAL, "nmodel must be >= 1");
    if (nlens < 0) return fail(LH_EINVAL, "nlens must be >= 0");
    if (nlens > 0 && !lenses) return fail(LH_EINVAL, "lenses is NULL");
    if ((long double)nmodel * nlens >= (long double)(1u << 30)) return fail(LH_EINVAL, "nmodel*nlens must be < 2^30");
    return check_grid(g, nmodel);
}

int eval_checked(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *o) {
    ctx.err[0] = 0;
    int rc = check_common(lenses, nmodel, nlens, g);
    if (rc) return rc;
    if (!o) return fail(LH_EINVAL, "outputs is NULL");
    double *p[NPLANES];
    planes_of(o, p);
    bool any = false;
    for (int k = 0; k < NPLANES; ++k) {
        if (!p[k]) continue;
        any = true;
        if ((rc = check_device_ptr(p[k], PLANE_NAMES[k]))) return rc;
    }
    if (!any) return fail(LH_EINVAL, "no output plane requested");
    return eval_device(lenses, nmodel, nlens, g, p);
}

}  // namespace

// What an entry point that lives in another file (lh_noalloc.cu) needs of this host thread's state: the stream of
// lh_set_stream, the text behind lh_last_error and the counter behind lh_launch_count.
namespace lh {
cudaStream_t api_stream() { return ctx.stream; }
int api_fail(int code, const char *msg) { return fail(code, "%s", msg); }
void api_clear_error() { ctx.err[0] = 0; }
long long *api_launch_counter() { return &ctx.launches; }
}  // namespace lh

extern "C" {

int lh_grid_eval(const lh_lens *lenses, int nlens, const lh_grid *g, const lh_outputs *o) {
    return eval_checked(lenses, 1, nlens, g, o);
}

int lh_grid_eval_rows(const lh_lens *lenses, int nlens, const lh_grid *g, int j0, int nrows, const lh_outputs *o) {
    ctx.err[0] = 0;
    int rc = check_common(lenses, 1, nlens, g);
    if (rc) return rc;
    if (j0 < 0 || nrows < 1 || (long long)j0 + nrows > g->ny) return fail(LH_EINVAL, "row slab outside the grid");
    if (!o) return fail(LH_EINVAL, "outputs is NULL");
    double *p[NPLANES];
    planes_of(o, p);
    bool any = false;
    for (int k = 0; k < NPLANES; ++k) {
        if (!p[k]) continue;
        any = true;
        if ((rc = check_device_ptr(p[k], PLANE_NAMES[k]))) return rc;
    }
    if (!any) return fail(LH_EINVAL, "no output plane requested");
    // the slab planes are stand-alone buffers: present them as a grid of nrows rows whose row 0 is grid row j0
    lh_grid slab = *g;
    slab.ny = nrows;
    EvalOpts opt;
    opt.j0 = j0; opt.nrows = nrows;
    return eval_device(lenses, 1, nlens, &slab, p, opt);
}

int lh_points_eval(const lh_lens *lenses, int nlens, const double *xs, const double *ys, long long npoints,
                   const lh_outputs *o) {
    ctx.err[0] = 0;
    if (npoints < 1 || npoints > 0x7fffffffLL) return fail(LH_EINVAL, "npoints must be in [1, 2^31)");
    if (!xs || !ys) return fail(LH_EINVAL, "lh_points_eval: xs and ys are required");
    lh_grid g = {0.0, 0.0, 1.0, (int32_t)npoints, 1};  // one row of "pixels"; the coordinates come from xs, ys
    int rc = check_common(lenses, 1, nlens, &g);
    if (rc) return rc;
    if ((rc = check_device_ptr(xs, "xs")) || (rc = check_device_ptr(ys, "ys"))) return rc;
    if (!o) return fail(LH_EINVAL, "outputs is NULL");
    double *p[NPLANES];
    planes_of(o, p);
    bool any = false;
    for (int k = 0; k < NPLANES; ++k) {
        if (!p[k]) continue;
        any = true;
        if ((rc = check_device_ptr(p[k], PLANE_NAMES[k]))) return rc;
    }
    if (!any) return fail(LH_EINVAL, "no output plane requested");
    EvalOpts opt;
    opt.px = xs; opt.py = ys;
    return eval_device(lenses, 1, nlens, &g, p, opt);
}

int lh_grid_eval_batch(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *o) {
    return eval_checked(lenses, nmodel, nlens, g, o);
}

int lh_grid_gradient(const lh_lens *lenses, int nlens, const lh_grid *g, double *out_ax, double *out_ay) {
    if (!out_ax || !out_ay) return fail(LH_EINVAL, "lh_grid_gradient: out_ax and out_ay are required");
    lh_outputs o;
    std::memset(&o, 0, sizeof(o));
    o.ax = out_ax; o.ay = out_ay;
    return eval_checked(lenses, 1, nlens, g, &o);
}

int lh_grid_hessian(const lh_lens *lenses, int nlens, const lh_grid *g, double *a11, double *a12, double *a22) {
    if (!a11 || !a12 || !a22) return fail(LH_EINVAL, "lh_grid_hessian: a11, a12 and a22 are required");
    lh_outputs o;
    std::memset(&o, 0, sizeof(o));
    o.a11 = a11; o.a12 = a12; o.a22 = a22;
    return eval_checked(lenses, 1, nlens, g, &o);
}

int lh_lens_maps(const lh_lens *lenses, int nlens, const lh_grid *g, double *kappa, double *gamma1, double *gamma2,
                 double *mu) {
    if (!kappa || !gamma1 || !gamma2 || !mu) return fail(LH_EINVAL, "lh_lens_maps: all four planes are required");
    lh_outputs o;
    std::memset(&o, 0, sizeof(o));
    o.kappa = kappa; o.gamma1 = gamma1; o.gamma2 = gamma2; o.mu = mu;
    return eval_checked(lenses, 1, nlens, g, &o);
}

int lh_grid_gradient_batch(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, double *out_ax,
                           double *out_ay) {
    if (!out_ax || !out_ay) return fail(LH_EINVAL, "lh_grid_gradient_batch: out_ax and out_ay are required");
    lh_outputs o;
    std::memset(&o, 0, sizeof(o));
    o.ax = out_ax; o.ay = out_ay;
    return eval_checked(lenses, nmodel, nlens, g, &o);
}

int lh_grid_eval_batch_shared(const lh_lens *shared, int nshared, const lh_lens *varying, int nmodel, int nvar,
                              const lh_grid *g, const lh_outputs *o) {
    ctx.err[0] = 0;
    int rc = check_common(varying, nmodel, nvar, g);
    if (rc) return rc;
    if (nshared < 0 || (nshared > 0 && !shared)) return fail(LH_EINVAL, "shared lens list: bad argument");
    if (nshared >= (1 << 30)) return fail(LH_EINVAL, "nshared must be < 2^30");
    if (nshared > 0 && nvar > lh::LAUNCH_RECORDS)
        return fail(LH_EINVAL, "at most %d varying lenses per model beside a shared list", lh::LAUNCH_RECORDS);
    if (!o) return fail(LH_EINVAL, "outputs is NULL");
    double *p[NPLANES];
    planes_of(o, p);
    bool any = false;
    for (int k = 0; k < NPLANES; ++k) {
        if (!p[k]) continue;
        any = true;
        if ((rc = check_device_ptr(p[k], PLANE_NAMES[k]))) return rc;
    }
    if (!any) return fail(LH_EINVAL, "no output plane requested");
    EvalOpts opt;
    opt.shared = shared; opt.nshared = nshared;
    return eval_device(varying, nmodel, nvar, g, p, opt);
}

int lh_grid_stats_batch(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *mean,
                        const lh_outputs *var) {
    ctx.err[0] = 0;
    int rc = check_common(lenses, nmodel, nlens, g);
    if (rc) return rc;
    if ((rc = check_grid(g, 1))) return rc;
    if (!mean) return fail(LH_EINVAL, "lh_grid_stats_batch: mean is NULL");
    double *pm[NPLANES], *pv[NPLANES];
    planes_of(mean, pm);
    for (int k = 0; k < NPLANES; ++k) pv[k] = nullptr;
    if (var) planes_of(var, pv);
    bool any = false;
    for (int k = 0; k < NPLANES; ++k) {
        if (pv[k] && !pm[k]) return fail(LH_EINVAL, "variance of %s requested without its mean", PLANE_NAMES[k]);
        if (pm[k]) {
            any = true;
            if ((rc = check_device_ptr(pm[k], PLANE_NAMES[k]))) return rc;
        }
        if (pv[k] && (rc = check_device_ptr(pv[k], PLANE_NAMES[k]))) return rc;
        if (pv[k] && pv[k] == pm[k]) return fail(LH_EINVAL, "mean and variance of %s share a buffer", PLANE_NAMES[k]);
    }
    if (!any) return fail(LH_EINVAL, "no output plane requested");
    EvalOpts opt;
    opt.m2 = pv;
    return eval_device(lenses, nmodel, nlens, g, pm, opt);
}

int lh_source_plane(const double *ax, const double *ay, const lh_grid *g, double *bx, double *by) {
    ctx.err[0] = 0;
    int rc = check_grid(g, 1);
    if (rc) return rc;
    if (!ax || !ay) return fail(LH_EINVAL, "lh_source_plane: ax and ay are required");
    if (!bx && !by) return fail(LH_EINVAL, "no output plane requested");
    if ((rc = check_device_ptr(ax, "ax")) || (rc = check_device_ptr(ay, "ay"))) return rc;
    if (bx && (rc = check_device_ptr(bx, "bx"))) return rc;
    if (by && (rc = check_device_ptr(by, "by"))) return rc;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CU(lh::launch_source_plane(ax, ay, g->x0, g->y0, g->dx, g->nx, g->ny, bx, by, sms, ctx.stream));
    ++ctx.launches;
    return LH_OK;
}

int lh_delens_grid(const double *ax, const double *ay, const lh_grid *g, const double *sources, int nsources,
                   lh_image *images, long long max_images, long long *count) {
    ctx.err[0] = 0;
    int rc = check_grid(g, 1);
    if (rc) return rc;
    if (!ax || !ay || !count) return fail(LH_EINVAL, "lh_delens_grid: ax, ay and count are required");
    if (nsources < 0 || max_images < 0) return fail(LH_EINVAL, "lh_delens_grid: nsources and max_images must be >= 0");
    if (nsources > 0 && !sources) return fail(LH_EINVAL, "sources is NULL");
    if (max_images > 0 && !images) return fail(LH_EINVAL, "images is NULL");
    if ((rc = check_device_ptr(ax, "ax")) || (rc = check_device_ptr(ay, "ay"))) return rc;
    if ((rc = check_device_ptr(reinterpret_cast<const double *>(count), "count"))) return rc;
    if (images && (rc = check_device_ptr(reinterpret_cast<const double *>(images), "images"))) return rc;
    for (int s = 0; s < 2 * nsources; ++s)
        if (!std::isfinite(sources[s])) return fail(LH_EINVAL, "source %d: non-finite position", s / 2);
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CU(cudaMemsetAsync(count, 0, sizeof(long long), ctx.stream));
    CU(lh::launch_delens(ax, ay, g->x0, g->y0, g->dx, g->nx, g->ny, sources, nsources, images, max_images,
                         reinterpret_cast<unsigned long long *>(count), sms, ctx.stream, &ctx.launches));
    return LH_OK;
}

int lh_chi2(const lh_lens *lenses, int nlens, const lh_grid *g, const lh_constraint *constraints, int nconstraints,
            int nsources, double *chi2, double *predicted, double *sources, long long *nimages) {
    ctx.err[0] = 0;
    int rc = check_common(lenses, 1, nlens, g);
    if (rc) return rc;
    const int K = nconstraints, N = nsources;
    if (K < 0 || N < 0 || (K > 0 && !constraints)) return fail(LH_EINVAL, "lh_chi2: bad constraint list");
    if (!chi2) return fail(LH_EINVAL, "lh_chi2: chi2 is required");
    for (int k = 0; k < K; ++k) {
        const lh_constraint &c = constraints[k];
        if (c.source < 0 || c.source >= N) return fail(LH_EINVAL, "constraint %d: source index outside [0, nsources)", k);
        if (!(std::isfinite(c.x) && std::isfinite(c.y) && std::isfinite(c.sigma)) || !(c.sigma > 0.0))
            return fail(LH_EINVAL, "constraint %d: non-finite position or sigma <= 0", k);
    }
    if ((rc = check_device_ptr(chi2, "chi2"))) return rc;
    if (predicted && (rc = check_device_ptr(predicted, "predicted"))) return rc;
    if (sources && (rc = check_device_ptr(sources, "sources"))) return rc;
    if (nimages && (rc = check_device_ptr(reinterpret_cast<double *>(nimages), "nimages"))) return rc;
    // validate and pack the lens list once; both evaluations below reuse the packed table
    if ((rc = pack_all(lenses, 1, nlens))) return rc;

    // scratch layout (all 16-byte aligned)
    const size_t npix = (size_t)g->nx * g->ny;
    const long long cap = 64LL * K + 4096;
    auto al = [](size_t b) { return (b + 15) & ~size_t(15); };
    const size_t o_ax = 0, o_ay = o_ax + al(npix * 8), o_c = o_ay + al(npix * 8), o_cx = o_c + al((size_t)K * 32 + 16),
                 o_cy = o_cx + al((size_t)K * 8 + 16), o_bax = o_cy + al((size_t)K * 8 + 16),
                 o_bay = o_bax + al((size_t)K * 8 + 16), o_term = o_bay + al((size_t)K * 8 + 16),
                 o_src = o_term + al((size_t)K * 8 + 16), o_cnt = o_src + al((size_t)N * 16 + 16), o_im = o_cnt + 16,
                 total = o_im + (size_t)cap * sizeof(lh_image);
    cudaStream_t s = ctx.stream;
    // Everything that can fail for lack of memory is obtained BEFORE the first enqueue: the scratch buffer, the carry
    // buffer of the larger of the two evaluations and the math tables.  The scratch is cached per device and reused
    // across calls: stream order protects it on one stream, ev_chi + cudaStreamWaitEvent across a stream change, and
    // it is only freed after the last call that used it has finished.
    if (!DS().ev_chi) CU(cudaEventCreateWithFlags(&DS().ev_chi, cudaEventDisableTiming));
    if (total > DS().chi_bytes) {
        if (DS().d_chi) {
            if (DS().chi_busy) CU(cudaEventSynchronize(DS().ev_chi));
            cudaFree(DS().d_chi);
            DS().d_chi = nullptr;
            DS().chi_bytes = 0;
            DS().chi_busy = false;
        }
        CU(cudaMalloc(&DS().d_chi, total));
        DS().chi_bytes = total;
    }
    if (DS().chi_busy && DS().chi_stream != s) CU(cudaStreamWaitEvent(s, DS().ev_chi, 0));
    if (nlens > lh::LAUNCH_RECORDS) {
        const size_t big = npix > (size_t)K ? npix : (size_t)K;
        if ((rc = ensure_carry((size_t)5 * big * sizeof(double), s))) return rc;
        if ((rc = ensure_aux_stream())) return rc;  // stage 1 runs its row halves as two chains (eval_device)
    }
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    {
        cudaError_t terr;
        if (!device_math_tables(dev, &terr)) return fail(LH_ECUDA, "math tables: %s", cudaGetErrorString(terr));
    }
    char *B = DS().d_chi;
    double *ax = reinterpret_cast<double *>(B + o_ax), *ay = reinterpret_cast<double *>(B + o_ay);
    lh_constraint *dc = reinterpret_cast<lh_constraint *>(B + o_c);
    double *cx = reinterpret_cast<double *>(B + o_cx), *cy = reinterpret_cast<double *>(B + o_cy);
    double *bax = reinterpret_cast<double *>(B + o_bax), *bay = reinterpret_cast<double *>(B + o_bay);
    double *term = reinterpret_cast<double *>(B + o_term);
    double *src = sources ? sources : reinterpret_cast<double *>(B + o_src);
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(B + o_cnt);
    lh_image *im = reinterpret_cast<lh_image *>(B + o_im);
    EvalOpts packed;
    packed.packed0 = 0;

    // stage 2: unlens the constraints at their own positions, barycentre per source
    if (K > 0) {
        CU(cudaMemcpyAsync(dc, constraints, (size_t)K * sizeof(lh_constraint), cudaMemcpyHostToDevice, s));
        CU(lh::launch_constraint_points(dc, K, cx, cy, s));
        ++ctx.launches;
        lh_grid pg = {0.0, 0.0, 1.0, K, 1};
        double *po[NPLANES] = {bax, bay, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
        EvalOpts opt = packed;
        opt.px = cx; opt.py = cy;
        if ((rc = eval_device(lenses, 1, nlens, &pg, po, opt))) return rc;
    }
    CU(lh::launch_barycentre(dc, K, bax, bay, N, src, s));
    ++ctx.launches;
    // stage 1: deflection on the grid
    double *go[NPLANES] = {ax, ay, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    if ((rc = eval_device(lenses, 1, nlens, g, go, packed))) return rc;
    // stage 3: predicted images
    CU(cudaMemsetAsync(cnt, 0, sizeof(*cnt), s));
    CU(lh::launch_delens_dev(ax, ay, g->x0, g->y0, g->dx, g->nx, g->ny, src, N, im, cap, cnt, sms, s, &ctx.launches));
    // stage 4: closest image of the same source, chi^2
    CU(lh::launch_assign_and_sum(dc, K, im, cnt, cap, predicted, term, chi2, nimages, s));
    ctx.launches += (K > 0) + 1;
    CU(cudaEventRecord(DS().ev_chi, s));
    DS().chi_busy = true;
    DS().chi_stream = s;
    return LH_OK;
}

}  // extern "C"

namespace {

// HOST output planes.  One map (nmodel == 1): rows [j0, j0 + nrows) of the grid into planes of nrows x nx doubles;
// a batch: all rows of every model.
// Host copy of one piece out of the pinned ring into the caller's pageable planes, on a few threads (one thread
// moves 8-12 GB/s; the step would otherwise wait for it).
void parallel_copy(char *dst, const char *src, size_t bytes) {
    unsigned hw = std::thread::hardware_concurrency();
    const int nt = (int)std::min<size_t>(hw ? (hw > 8 ? 8 : hw) : 1, bytes / (4u << 20) + 1);
    if (nt <= 1) { std::memcpy(dst, src, bytes); return; }
    // No exception may cross the C ABI (lh.h) and a joinable std::thread must never be destroyed: the helpers live in
    // a fixed array (no allocation that could throw between two spawns), and a spawn that fails (EAGAIN under a pid
    // limit) leaves its share, and every share after it, to the calling thread.
    std::thread th[8];
    int started = 0;
    const size_t per = ((bytes / nt) + 4095) & ~size_t(4095);
    size_t done_to = per < bytes ? per : bytes;  // the calling thread copies [0, per) and whatever no helper took
    for (int t = 1; t < nt && t <= 8; ++t) {
        const size_t o = per * t;
        if (o >= bytes) break;
        const size_t n = bytes - o < per ? bytes - o : per;
        try {
            th[started] = std::thread([=] { std::memcpy(dst + o, src + o, n); });
        } catch (...) {
            break;
        }
        ++started;
        done_to = o + n;
    }
    std::memcpy(dst, src, per < bytes ? per : bytes);
    if (done_to < bytes) std::memcpy(dst + done_to, src + done_to, bytes - done_to);
    for (int t = 0; t < started; ++t) th[t].join();
}

int eval_host(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, int j0, int nrows, const lh_outputs *host_o) {
    ctx.err[0] = 0;
    int rc = check_common(lenses, nmodel, nlens, g);
    if (rc) return rc;
    if (j0 < 0 || nrows < 1 || (long long)j0 + nrows > g->ny) return fail(LH_EINVAL, "row slab outside the grid");
    if (nmodel > 1 && (j0 != 0 || nrows != g->ny)) return fail(LH_EINVAL, "row slabs of a batch are not supported");
    if (!host_o) return fail(LH_EINVAL, "outputs is NULL");
    double *hp[NPLANES], *dp[NPLANES];
    planes_of(host_o, hp);
    int nreq = 0;
    for (int k = 0; k < NPLANES; ++k) nreq += hp[k] != nullptr;
    if (!nreq) return fail(LH_EINVAL, "no output plane requested");
    // validate and pack every model ONCE, before anything is enqueued or copied (LH_EINVAL: nothing written); the
    // pieces below reuse the packed table
    if ((rc = pack_all(lenses, nmodel, nlens))) return rc;
    const size_t plane_bytes = (size_t)nmodel * g->nx * nrows * sizeof(double);
    const size_t need = plane_bytes * nreq;
    if (need > DS().planes_bytes) {
        if (DS().d_planes) {
            CU(cudaStreamSynchronize(ctx.stream));
            cudaFree(DS().d_planes);
            DS().d_planes = nullptr;
            DS().planes_bytes = 0;
        }
        CU(cudaMalloc(&DS().d_planes, need));
        DS().planes_bytes = need;
    }
    int slot = 0;
    for (int k = 0; k < NPLANES; ++k)
        dp[k] = hp[k] ? DS().d_planes + (size_t)(slot++) * (plane_bytes / sizeof(double)) : nullptr;
#ifdef LH_BOUNDS_CHECK
    // the internal device planes of this call, exactly as large as the call needs them (popped again below)
    struct PopRange { ~PopRange() { --dbg.n; } } pop_range;
    if (dbg.n >= lh::DBG_RANGES - 2) { ++dbg.n; return fail(LH_EINVAL, "too many debug ranges"); }
    dbg.lo[dbg.n] = reinterpret_cast<const char *>(DS().d_planes);
    dbg.hi[dbg.n] = reinterpret_cast<const char *>(DS().d_planes) + need;
    ++dbg.n;
#endif

    // Pipeline: the work is cut into pieces (row slabs of one map, or groups of models of a batch); the
    // device-to-host copy of piece k runs on a second stream while piece k+1 is being computed.
    if (!DS().copy_stream) {
        CU(cudaStreamCreateWithFlags(&DS().copy_stream, cudaStreamNonBlocking));
        for (int k = 0; k < DeviceState::PIECES; ++k) {
            CU(cudaEventCreateWithFlags(&DS().ev_piece[k], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&DS().ev_copied[k], cudaEventDisableTiming));
        }
    }
    // Pageable host planes: a device-to-pageable cudaMemcpyAsync is staged by the driver at about 6 GB/s and would BE the
    // step (cfg 3: 139 ms against 84 ms of computing).  Such planes are served through a pinned ring of two slots
    // instead: piece k is copied device -> ring at link speed while piece k+1 computes, and host threads move it
    // ring -> caller's planes meanwhile.  Pinned (or registered) planes are written directly.
    bool pageable = false;
    for (int k = 0; k < NPLANES; ++k) {
        if (!hp[k]) continue;
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, hp[k]) != cudaSuccess) { cudaGetLastError(); pageable = true; }
        else if (at.type == cudaMemoryTypeUnregistered) pageable = true;
    }
    const size_t npix = (size_t)g->nx * g->ny;
    const int units = nmodel == 1 ? nrows : nmodel;  // rows or models
    // the device planes of one map hold the slab only: present it as a grid of `nrows` rows whose row 0 is grid row j0
    lh_grid slab = *g;
    if (nmodel == 1) slab.ny = nrows;
    // small jobs are not worth cutting: about 4 MB of results per piece at least
    long long want = (long long)(need >> 22);
    const int pieces = want < 1 ? 1 : (want > DeviceState::PIECES ? DeviceState::PIECES : (int)want);
    int per = (units + pieces - 1) / pieces;
    if (nmodel == 1) per = (per + 7) & ~7;            // whole pixel tiles
    const size_t piece_elems = nmodel == 1 ? (size_t)per * g->nx : (size_t)per * npix;  // per plane, at most
    const size_t slot_bytes = piece_elems * sizeof(double) * nreq;
    if (pageable && 2 * slot_bytes > DS().ring_bytes) {
        if (DS().h_ring) {
            CU(cudaStreamSynchronize(DS().copy_stream));
            cudaFreeHost(DS().h_ring);
            DS().h_ring = nullptr;
            DS().ring_bytes = 0;
        }
        CU(cudaMallocHost(&DS().h_ring, 2 * slot_bytes));
        DS().ring_bytes = 2 * slot_bytes;
    }
    // One map: the pieces are independent (disjoint rows of the planes AND of the carry buffer), so the odd ones go to
    // a second stream and the part-filled last wave of one piece's launches is filled by the next piece's CTAs.
    // (Not with pageable planes: there the host drains piece k-1 before it enqueues piece k+1, and two pieces sharing
    // the GPU would make it wait longer for k-1 and starve the queue -- measured 96.8 ms against 91.6.)
    const bool two_streams = nmodel == 1 && pieces > 1 && !pageable;
    cudaStream_t user_stream = ctx.stream;
    if (two_streams) {
        if (!DS().piece_stream) {
            CU(cudaStreamCreateWithFlags(&DS().piece_stream, cudaStreamNonBlocking));
            CU(cudaEventCreateWithFlags(&DS().ev_pfork, cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&DS().ev_pjoin, cudaEventDisableTiming));
        }
        if (nlens > lh::LAUNCH_RECORDS && (rc = ensure_carry((size_t)5 * g->nx * nrows * sizeof(double), user_stream))) return rc;
        CU(cudaEventRecord(DS().ev_pfork, user_stream));
        CU(cudaStreamWaitEvent(DS().piece_stream, DS().ev_pfork, 0));
    }
    // ring -> caller's planes for piece q (blocks until its device -> ring copies have landed)
    struct Pending { size_t off, count; int slot; bool live; } pend = {0, 0, 0, false};
    auto drain = [&](int q) -> int {
        if (!pend.live) return LH_OK;
        CU(cudaEventSynchronize(DS().ev_copied[q]));
        int s = 0;
        for (int k = 0; k < NPLANES; ++k) {
            if (!hp[k]) continue;
            parallel_copy(reinterpret_cast<char *>(hp[k] + pend.off),
                          DS().h_ring + (size_t)pend.slot * slot_bytes + (size_t)s * piece_elems * sizeof(double),
                          pend.count * sizeof(double));
            ++s;
        }
        pend.live = false;
        return LH_OK;
    };
    // The pieces, as one unit that may stop early: whatever it returns, the epilogue below joins the streams, hands
    // the carry buffer back and waits for everything that was enqueued (a failure on a later piece must not leave
    // piece_stream unjoined or kernels running on a carry buffer the next call might free).
    auto pipeline = [&]() -> int {
    int rc = LH_OK;
    int piece = 0;
    for (int u0 = 0; u0 < units; u0 += per, ++piece) {
        const int nu = units - u0 < per ? units - u0 : per;
        double *sub[NPLANES];
        const size_t off = nmodel == 1 ? (size_t)u0 * g->nx : (size_t)u0 * npix;
        const size_t count = nmodel == 1 ? (size_t)nu * g->nx : (size_t)nu * npix;
        for (int k = 0; k < NPLANES; ++k) sub[k] = dp[k] ? dp[k] + off : nullptr;
        EvalOpts opt;
        if (nmodel == 1) { opt.j0 = j0 + u0; opt.nrows = nu; opt.buf_row0 = u0; opt.packed0 = 0; }
        else opt.packed0 = u0;
        cudaStream_t pstream = user_stream;
        if (two_streams) {
            pstream = (piece & 1) ? DS().piece_stream : user_stream;
            opt.stream_override = pstream;
            opt.carry_guard_by_caller = true;
        }
        rc = eval_device(lenses, nmodel == 1 ? 1 : nu, nlens, nmodel == 1 ? &slab : g, sub, opt);
        if (rc) return rc;  // only a CUDA failure can get here: the lens lists were validated above
        CU(cudaEventRecord(DS().ev_piece[piece], pstream));
        CU(cudaStreamWaitEvent(DS().copy_stream, DS().ev_piece[piece], 0));
        if (!pageable) {
            for (int k = 0; k < NPLANES; ++k)
                if (hp[k]) CU(cudaMemcpyAsync(hp[k] + off, dp[k] + off, count * sizeof(double), cudaMemcpyDeviceToHost, DS().copy_stream));
            continue;
        }
        // slot piece % 2 is free: the piece that used it last (piece - 2) was drained during the previous iteration
        int s = 0;
        for (int k = 0; k < NPLANES; ++k) {
            if (!hp[k]) continue;
            CU(cudaMemcpyAsync(DS().h_ring + (size_t)(piece & 1) * slot_bytes + (size_t)s * piece_elems * sizeof(double), dp[k] + off,
                               count * sizeof(double), cudaMemcpyDeviceToHost, DS().copy_stream));
            ++s;
        }
        CU(cudaEventRecord(DS().ev_copied[piece], DS().copy_stream));
        if ((rc = drain(piece - 1))) return rc;  // the PREVIOUS piece, while this one computes and copies
        pend = {off, count, piece & 1, true};
    }
    if (pageable && (rc = drain(piece - 1))) return rc;
    return LH_OK;
    };
    rc = pipeline();
    // epilogue, after success and failure alike; the FIRST error keeps its message
    int rc2 = LH_OK;
    auto keep = [&](cudaError_t e, const char *what) {
        if (e != cudaSuccess && rc == LH_OK && rc2 == LH_OK) rc2 = fail(LH_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    };
    if (two_streams) {  // join, and hand the carry buffer back to the ordinary one-stream protocol
        keep(cudaEventRecord(DS().ev_pjoin, DS().piece_stream), "cudaEventRecord(ev_pjoin)");
        keep(cudaStreamWaitEvent(user_stream, DS().ev_pjoin, 0), "cudaStreamWaitEvent(ev_pjoin)");
        if (nlens > lh::LAUNCH_RECORDS) {
            keep(cudaEventRecord(DS().ev_done, user_stream), "cudaEventRecord(ev_done)");
            DS().busy = true;
            DS().last_stream = user_stream;
        }
    }
    keep(cudaStreamSynchronize(DS().copy_stream), "cudaStreamSynchronize(copy stream)");
    keep(cudaStreamSynchronize(ctx.stream), "cudaStreamSynchronize");
    pend.live = false;  // nothing is in flight any more: a ring slot with an undrained piece is simply abandoned
    return rc ? rc : rc2;
}

}  // namespace

extern "C" {

int lh_grid_eval_host(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *host_o) {
    return eval_host(lenses, nmodel, nlens, g, 0, g ? g->ny : 0, host_o);
}

int lh_grid_eval_rows_host(const lh_lens *lenses, int nlens, const lh_grid *g, int j0, int nrows, const lh_outputs *host_o) {
    return eval_host(lenses, 1, nlens, g, j0, nrows, host_o);
}

int lh_pack_model(const lh_lens *lenses, int n, double *table, int32_t *class_begin) {
    static_assert(LH_PACK_DOUBLES == lh::LENSK_DOUBLES && LH_PACK_CLASSES == lh::CLS_COUNT, "lh.h out of date");
    ctx.err[0] = 0;
    if (n < 0 || (n > 0 && !lenses) || !class_begin) return fail(LH_EINVAL, "lh_pack_model: bad argument");
    LensK *tmp = table ? reinterpret_cast<LensK *>(table) : new (std::nothrow) LensK[n > 0 ? n : 1];
    if (!tmp) return fail(LH_EINVAL, "lh_pack_model: out of memory");
    if (table && (reinterpret_cast<uintptr_t>(table) & 15u)) return fail(LH_EINVAL, "table must be 16-byte aligned");
    ModelRanges r;
    const int rc = lh::pack_model(lenses, n, tmp, &r, ctx.err, sizeof(ctx.err), 0);
    if (!table) delete[] tmp;
    if (rc != 0) return LH_EINVAL;
    for (int k = 0; k <= lh::CLS_COUNT; ++k) class_begin[k] = r.begin[k];
    return LH_OK;
}

// ---- CUDA IPC wrappers (include/lh.h: a rank's slab written straight into the owner's map) -----------------------
namespace {
struct IpcMapping { void *user; void *base; };
std::mutex ipc_mu;
std::vector<IpcMapping> ipc_open_list;
}  // namespace

int lh_ipc_export(const void *dev_ptr, unsigned char handle[LH_IPC_HANDLE_BYTES], unsigned long long *offset) {
    static_assert(sizeof(cudaIpcMemHandle_t) == LH_IPC_HANDLE_BYTES, "lh.h out of date");
    ctx.err[0] = 0;
    if (!dev_ptr || !handle || !offset) return fail(LH_EINVAL, "lh_ipc_export: NULL argument");
    int rc = check_device_ptr(static_cast<const double *>(dev_ptr), "dev_ptr");
    if (rc) return rc;
    // base of the allocation that holds dev_ptr (driver entry point fetched at run time: no link-time libcuda)
    typedef int (*range_fn)(unsigned long long *, size_t *, unsigned long long);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    CU(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qr));
    if (!fn || qr != cudaDriverEntryPointSuccess) return fail(LH_ECUDA, "cuMemGetAddressRange is not available");
    unsigned long long base = 0;
    size_t size = 0;
    if (reinterpret_cast<range_fn>(fn)(&base, &size, (unsigned long long)reinterpret_cast<uintptr_t>(dev_ptr)) != 0)
        return fail(LH_EINVAL, "lh_ipc_export: not the address of a device allocation");
    cudaIpcMemHandle_t h;
    CU(cudaIpcGetMemHandle(&h, reinterpret_cast<void *>(static_cast<uintptr_t>(base))));
    std::memcpy(handle, &h, sizeof(h));
    *offset = (unsigned long long)reinterpret_cast<uintptr_t>(dev_ptr) - base;
    return LH_OK;
}

int lh_ipc_open(const unsigned char handle[LH_IPC_HANDLE_BYTES], unsigned long long offset, void **dev_ptr) {
    ctx.err[0] = 0;
    if (!handle || !dev_ptr) return fail(LH_EINVAL, "lh_ipc_open: NULL argument");
    cudaIpcMemHandle_t h;
    std::memcpy(&h, handle, sizeof(h));
    void *base = nullptr;
    CU(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    *dev_ptr = static_cast<char *>(base) + offset;
    std::lock_guard<std::mutex> lock(ipc_mu);
    ipc_open_list.push_back(IpcMapping{*dev_ptr, base});
    return LH_OK;
}

int lh_ipc_close(void *dev_ptr) {
    ctx.err[0] = 0;
    void *base = nullptr;
    {
        std::lock_guard<std::mutex> lock(ipc_mu);
        for (size_t k = 0; k < ipc_open_list.size(); ++k)
            if (ipc_open_list[k].user == dev_ptr) {
                base = ipc_open_list[k].base;
                ipc_open_list.erase(ipc_open_list.begin() + (long)k);
                break;
            }
    }
    if (!base) return fail(LH_EINVAL, "lh_ipc_close: not a pointer lh_ipc_open returned");
    CU(cudaIpcCloseMemHandle(base));
    return LH_OK;
}

#ifdef LH_BOUNDS_CHECK
// ---- checking build only; not declared in include/lh.h (tests/test_gpu_bounds.py declares them itself) -------------
int lh_debug_bounds_reset(void) {
    dbg.n = 0;
    if (dbg.d_count) {
        CU(cudaDeviceSynchronize());
        CU(cudaMemset(dbg.d_count, 0, sizeof(unsigned long long)));
    }
    return LH_OK;
}
int lh_debug_bounds_add(const void *p, unsigned long long bytes) {
    if (!p || dbg.n >= lh::DBG_RANGES - 2) return fail(LH_EINVAL, "lh_debug_bounds_add: NULL or too many ranges");
    dbg.lo[dbg.n] = static_cast<const char *>(p);
    dbg.hi[dbg.n] = static_cast<const char *>(p) + bytes;
    ++dbg.n;
    return LH_OK;
}
long long lh_debug_violations(void) {
    if (!dbg.d_count) return 0;
    unsigned long long v = 0;
    if (cudaDeviceSynchronize() != cudaSuccess) return -1;
    if (cudaMemcpy(&v, dbg.d_count, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    return (long long)v;
}
#endif

int lh_set_stream(void *cuda_stream) {
    ctx.stream = static_cast<cudaStream_t>(cuda_stream);
    return LH_OK;
}

const char *lh_last_error(void) { return ctx.err; }

long long lh_launch_count(void) { return ctx.launches; }

int lh_fp64_peak_probe(int iters, double *flops_per_s, double *seconds) {
    ctx.err[0] = 0;
    if (iters <= 0 || !flops_per_s || !seconds) return fail(LH_EINVAL, "lh_fp64_peak_probe: bad argument");
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (!DS().d_sink) CU(cudaMalloc(&DS().d_sink, 64));
    const int blocks = sms * 8;  // 8 x 256 threads = 64 warps per SM
    cudaEvent_t t0, t1;
    CU(cudaEventCreate(&t0));
    CU(cudaEventCreate(&t1));
    CU(lh::launch_dfma_probe(iters / 8 + 1, blocks, DS().d_sink, ctx.stream));  // warm-up
    CU(cudaEventRecord(t0, ctx.stream));
    CU(lh::launch_dfma_probe(iters, blocks, DS().d_sink, ctx.stream));
    CU(cudaEventRecord(t1, ctx.stream));
    CU(cudaEventSynchronize(t1));
    ctx.launches += 2;
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, t0, t1));
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    const double fmas = (double)blocks * 256.0 * (double)iters * 64.0;
    *seconds = ms * 1e-3;
    *flops_per_s = 2.0 * fmas / (*seconds);
    return LH_OK;
}

int lh_math_host_eval(int fn, const double *a, const double *b, size_t n, double *out) {
    ctx.err[0] = 0;
    if (fn < 0 || fn > 6 || !a || !out || (fn >= 3 && !b)) return fail(LH_EINVAL, "lh_math_host_eval: bad argument");
    static lh::MathTables tab;
    static std::once_flag once;
    std::call_once(once, [] { lh::fill_math_tables(tab); });
    for (size_t k = 0; k < n; ++k) {
        double w, iw, i1, i2, i3, i4;
        switch (fn) {
            case 0: out[k] = lh::rcp(a[k]); break;
            case 1: lh::rsqrt_sqrt(a[k], w, iw); out[k] = w; break;
            case 2: lh::rsqrt_sqrt(a[k], w, iw); out[k] = iw; break;
            case 3: out[k] = lh::atan_nd(a[k], b[k], tab.at); break;
            case 4: out[k] = lh::atanh_nd(a[k], b[k], tab.ah); break;
            case 5: lh::rcp2(a[k], b[k], i1, i2); out[k] = i1; break;
            default: lh::rcp4(a[k], b[k], a[k] + b[k], 2.0 * b[k], i1, i2, i3, i4); out[k] = i1; break;
        }
    }
    return LH_OK;
}

const char *lh_version(void) { return "lh 0.1 sm_100a"; }

#ifndef LH_SOURCE_HASH
#define LH_SOURCE_HASH "unknown"
#endif
const char *lh_source_hash(void) { return LH_SOURCE_HASH; }

}  // extern "C"

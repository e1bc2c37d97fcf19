/*
 * lh.h -- C ABI of liblh.so: the lens-map hot path of Lenstool-HPC
 * (arXiv 2004.06352), built from scratch for NVIDIA B200 (sm_100a), FP64.
 *
 * What the library computes.  For every pixel of a regular image-plane grid
 * ("a rectangular grid defined on the image-plane, each grid cell usually being
 * the size of a pixel", PAPER.md:99 sec. 2.4; :181 sec. 4.1) and a list of N
 * parametric potentials (sec. 2.2):
 *
 *   - the deflection alpha = grad psi as the sum of the first derivatives of all
 *     potentials at that point (PAPER.md:183 eq. 10; :53 alpha = grad psi);
 *   - the second derivatives a_ij = d_ij psi, "at each grid-point the
 *     second-order derivative contribution of each cluster member is added up"
 *     (sec. 2.4);
 *   - the maps kappa = (a11+a22)/2, gamma1 = (a11-a22)/2, gamma2 = a12,
 *     mu = 1/((1-kappa)^2 - gamma1^2 - gamma2^2)
 *     (PAPER.md:57 eq. 4, :64 eq. 5, :105-110 eq. 7-9; garbled signs/sums read as
 *     DESIGN.md sec. 3 states).
 *
 * The paper does not print the potentials; the profiles (dPIE = difference of two
 * PIEMDs, NSIE, SIS), their normalisation and the ellipticity / angle conventions
 * are the readings listed in DESIGN.md sec. 3.
 *
 * Conventions common to every call
 *   units      arcsec for lengths, radians for theta; all reals IEEE binary64.
 *   lenses     HOST pointer, caller-owned, read only during the call (packed and
 *              copied before return; may be freed or changed right after).
 *   grid       HOST pointer, read during the call.
 *   outputs    DEVICE pointers (cudaMalloc / torch CUDA tensor .data_ptr()),
 *              caller-owned, 8-byte aligned, ny*nx doubles each (times nmodel for
 *              batch calls), row-major: pixel (i, j) at (x0 + i*dx, y0 + j*dx) is
 *              element j*nx + i; model m starts at m*ny*nx.  Fully overwritten.
 *              The *_host entry points take HOST pointers instead.
 *   stream     work is enqueued on the stream set by lh_set_stream() for the
 *              calling host thread (default: the legacy default stream) and the
 *              call returns without synchronising the device.  (The *_host entry
 *              points synchronise that stream before they return.)
 *   errors     0 on success, a negative code on failure; lh_last_error() gives a message.
 *              LH_EINVAL (a bad argument: every argument, every lens of every model and every
 *              constraint is checked first): nothing was enqueued, no output element written.
 *              LH_ECUDA (a CUDA call failed): work may already be enqueued; outputs undefined.
 *              No exception or abort crosses this boundary.
 *   nlens = 0  is valid: alpha = 0, a_ij = 0, kappa = gamma = 0, mu = 1.
 *   range      lengths (positions, radii, pixel size) may use any unit in which all of them lie between about
 *              1e-20 and 1e+17: the kernel takes ONE reciprocal of a product of two squared and two cubed lengths
 *              of the scaled lens frame (scale factor <= 2^40) per evaluation, and that
 *              product must stay inside the double range.
 *   IEEE       mu = +-inf where det A^-1 == 0 exactly.  A pixel that coincides
 *              exactly with the centre of an SIS gets zero contribution from it.
 */
#ifndef LH_H_
#define LH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LH_OK 0
#define LH_EINVAL (-1) /* bad argument; nothing was enqueued */
#define LH_ECUDA (-2)  /* a CUDA call failed; see lh_last_error() */

enum { LH_DPIE = 0, LH_NSIE = 1, LH_SIS = 2 };

/* One parametric potential, 64 bytes (AoS at the boundary; the library packs to a
 * per-lens table of precomputed constants, sorted by type, on the device). */
typedef struct {
    int32_t type;       /* LH_DPIE, LH_NSIE or LH_SIS */
    int32_t _pad;       /* ignored */
    double x, y;        /* centre */
    double ellipticity; /* e-hat = (A^2-B^2)/(A^2+B^2) of the mass isodensities, in [0,1); ignored for SIS */
    double theta;       /* position angle of the major axis, CCW from +x; ignored for SIS */
    double rcore;       /* dPIE: 0 < rcore < rcut; NSIE: > 0; SIS: ignored */
    double rcut;        /* dPIE only */
    double b0;          /* = (D_ls/D_s) 6 pi (sigma/c)^2 in arcsec, finite and >= 0 (SIS: |alpha| = b0) */
} lh_lens;

/* Regular grid with square pixels: pixel (i, j) at (x0 + i*dx, y0 + j*dx). */
typedef struct {
    double x0, y0, dx;
    int32_t nx, ny;
} lh_grid;

/* Up to nine output planes; NULL = not wanted (and then never touched). */
typedef struct {
    double *ax, *ay;                     /* deflection           (eq. 10) */
    double *a11, *a12, *a22;             /* Hessian of psi       (sec. 2.4) */
    double *kappa, *gamma1, *gamma2, *mu; /* maps                 (eq. 4, 5, 7-9) */
} lh_outputs;

/* alpha_x, alpha_y on the grid (eq. 10).  Both planes required.
 * LH_EINVAL: NULL pointer, nlens < 0, nx or ny <= 0, nx*ny >= 2^40, dx <= 0 or
 * non-finite x0/y0/dx, unknown lens type, non-finite parameter, b0 < 0, e-hat outside [0,1),
 * dPIE with rcore <= 0 or rcut <= rcore, NSIE with rcore <= 0, output pointer that
 * is not device memory or not 8-byte aligned. */
int lh_grid_gradient(const lh_lens *lenses, int nlens, const lh_grid *g, double *out_ax, double *out_ay);

/* a11 = d_xx psi, a12 = d_xy psi, a22 = d_yy psi summed over lenses.
 * All three planes required.  Errors as above. */
int lh_grid_hessian(const lh_lens *lenses, int nlens, const lh_grid *g, double *a11, double *a12, double *a22);

/* kappa, gamma1, gamma2, mu (PAPER.md:57-64 eq. 4-5; :105-110 eq. 7-9).  All four
 * planes required.  The Hessian is reduced in registers and never written. */
int lh_lens_maps(const lh_lens *lenses, int nlens, const lh_grid *g, double *kappa, double *gamma1, double *gamma2,
                 double *mu);

/* Deflection maps of `nmodel` lens models on one shared grid in one launch -- the
 * shape in which an MCMC sampler or the map-variance computation issues them
 * (PAPER.md:81 sec. 2.2; :101, :114 sec. 2.4).  lenses[m*nlens + l] is lens l of
 * model m; out_ax[m*ny*nx + j*nx + i].  nmodel >= 1, nmodel*nx*ny < 2^40. */
int lh_grid_gradient_batch(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, double *out_ax,
                           double *out_ay);

/* Any subset of the nine planes in ONE pass over the lenses (at least one plane
 * must be non-NULL).  The four calls above are thin wrappers of this one. */
int lh_grid_eval(const lh_lens *lenses, int nlens, const lh_grid *g, const lh_outputs *o);

/* Rows [j0, j0 + nrows) of the grid only -- the multi-GPU primitive: pixels are independent ("no need for
 * communication between the different parallel tasks"; the paper splits the grid among its GPUs,
 * PAPER.md:194), so each device evaluates a row slab with the whole lens list and no exchange.  The planes of
 * `o` hold nrows*nx doubles (row j0 first).  Pixel coordinates are those of the full grid, so the slab is
 * bit-identical to the same rows of lh_grid_eval.  0 <= j0, nrows >= 1, j0 + nrows <= ny. */
int lh_grid_eval_rows(const lh_lens *lenses, int nlens, const lh_grid *g, int j0, int nrows, const lh_outputs *o);

/* lh_grid_eval_rows for callers that must not allocate device memory.
 *
 * Who needs it.  The other entry points call cudaMalloc the first time they need their reduction tables and, for a
 * lens list longer than one launch carries (160 lenses), the `carry` planes that hand the partial sums of a pixel
 * from one launch to the next.  That is not acceptable to a program whose device memory is owned by someone else
 * (a framework's caching allocator or a scheduler that has taken the whole GPU: the library's cudaMalloc fails or
 * upsets the accounting), to a loop that must never stall (cudaMalloc / cudaFree synchronise the device), or where
 * the rule is "reserve everything at start-up".  This call makes NO cudaMalloc, cudaFree, stream, event or other
 * allocating CUDA call, and packs the lenses into a fixed host table: both buffers are `static __device__` arrays
 * inside liblh.so, reserved by the CUDA loader on every GPU that loads the library and held until the process ends.
 *
 * Limits (the price of a fixed reservation): nx*nrows <= LH_NOALLOC_MAX_PIXELS and nlens <= LH_NOALLOC_MAX_LENSES;
 * beyond either the call returns LH_EINVAL, says so in lh_last_error() and touches nothing.  A larger grid is
 * covered by several calls, one row slab each (slabs are bit-identical to the same rows of lh_grid_eval).
 * The reservation is 5 * LH_NOALLOC_MAX_PIXELS * 8 bytes = 40 MiB per GPU, plus 32 KB of tables.
 *
 * Arguments, layout, stream and result exactly as lh_grid_eval_rows: planes of nrows*nx doubles, row j0 first,
 * DEVICE pointers owned by the caller; enqueued on the lh_set_stream() stream as ONE launch chain (no second
 * stream), returns without synchronising.
 *
 * First call on each device: it looks up the device address of the two arrays (cudaGetSymbolAddress) and uploads
 * the tables with a synchronous cudaMemcpy.  Make that call once per device during set-up, with that device
 * current, and before any stream capture begins; later calls only pack and launch.
 *
 * One buffer for everybody.  Every call on a device uses the same scratch and leaves its last contents there.
 * Nothing needs clearing: the first launch of a chain starts its sums at zero without reading the scratch, and
 * every later launch reads only what the launch before it wrote for the same pixel.  For the same reason two calls
 * whose kernels can OVERLAP on the GPU (different streams, or different host threads on different streams) race on
 * it and produce garbage: keep the calls of one device on one stream, or order them with events.  Host-side the
 * call is serialised by a mutex, so calling from several threads is safe as long as the streams are ordered.
 * Not available in the checking build (liblh_check.so): LH_EINVAL there. */
#define LH_NOALLOC_MAX_PIXELS (1 << 20)
#define LH_NOALLOC_MAX_LENSES 4096
int lh_grid_eval_noalloc(const lh_lens *lenses, int nlens, const lh_grid *g, int j0, int nrows, const lh_outputs *o);

/* The same superposition at ARBITRARY points instead of a grid: xs, ys DEVICE [npoints]; every requested plane of
 * `o` holds npoints doubles.  (Stage 2 of the paper's chi^2 pipeline unlenses the observed images, which are not
 * on the grid: PAPER.md:76 Fig. 3, :192.)  Same kernels, same arithmetic; errors as lh_grid_gradient. */
int lh_points_eval(const lh_lens *lenses, int nlens, const double *xs, const double *ys, long long npoints,
                   const lh_outputs *o);

/* Batched form of lh_grid_eval (layout as lh_grid_gradient_batch). */
int lh_grid_eval_batch(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *o);

/* Batch whose models share most of their lenses (NEXT row f4): model m = `shared` (nshared lenses, the same for
 * every model -- e.g. the cluster galaxies an MCMC step leaves untouched) + varying[m*nvar .. (m+1)*nvar).  The
 * shared lenses are superposed ONCE; every model starts from those sums (the superposition is linear, PAPER.md:183
 * eq. 10, :112).  Result and layout as lh_grid_eval_batch on the concatenated lists (summation order differs).
 * nvar <= 160 when nshared > 0; nvar = 0 and nshared = 0 are valid.  Errors as lh_grid_gradient. */
int lh_grid_eval_batch_shared(const lh_lens *shared, int nshared, const lh_lens *varying, int nmodel, int nvar,
                              const lh_grid *g, const lh_outputs *o);

/* Per-pixel MEAN and VARIANCE of the requested planes over the `nmodel` lens models of a batch -- the
 * statistical-error maps of the Bayesian process: "In order to compute the map variances, full-resolution
 * lensing maps have to be generated for each tested parameter-combination" (sec. 2.4; 10014 maps
 * for Abell 2744).  No per-model map is materialised: every model's planes are reduced in
 * registers and folded into the running statistics (Welford) by the kernel epilogue, one launch chain per model
 * in model order.  mean->P / var->P are single [ny][nx] DEVICE planes; var may be NULL, and a variance plane
 * needs its mean plane.  Variance is the POPULATION variance (1/nmodel) sum (P_m - mean)^2 (R21).
 * mu is +-inf on critical lines, so its statistics are IEEE inf/NaN there.  Errors as lh_grid_gradient. */
int lh_grid_stats_batch(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *mean,
                        const lh_outputs *var);

/* ---- NEXT row f1: source plane and brute-force delensing ------------------------------------------------
 * Source-plane position of every grid pixel, beta = theta - alpha(theta) (eq. 1), from deflection
 * planes already on the device.  ax, ay, bx, by: DEVICE [ny][nx]; bx or by may be NULL (not wanted); bx / by may
 * alias ax / ay (in place).  Errors as lh_grid_gradient. */
int lh_source_plane(const double *ax, const double *ay, const lh_grid *g, double *bx, double *by);

/* One predicted image. */
typedef struct {
    int32_t source;   /* index into `sources` */
    int32_t _pad;     /* 0 */
    int64_t triangle; /* 2*(j*(nx-1)+i) + t: cell (i, j), t = 0 for (V00, V10, V01), 1 for (V11, V01, V10) */
    double x, y;      /* image-plane position */
} lh_image;

/* Brute-force image search: "unlens a image-plane grid unto the source-plane and check each quadrant for the
 * presence of the source" (sec. 2.3, Fig. 4; stage 3 of the chi^2 computation).
 * The grid pixels are the vertices; every cell is cut along V10-V01 into two triangles; a triangle whose
 * source-plane image contains source s (closed triangle, barycentric test) yields one image at the same
 * barycentric combination of its image-plane vertices (readings R22).
 *   ax, ay     DEVICE [ny][nx] deflection planes (e.g. from lh_grid_gradient on the same grid)
 *   sources    HOST [nsources][2] source-plane positions, read during the call
 *   images     DEVICE, room for max_images records; the ORDER of the records is not defined
 *   count      DEVICE; set to the number of images FOUND, which may exceed max_images (then only
 *              max_images records were stored)
 * Asynchronous on the set stream.  LH_EINVAL: NULL pointer, nsources < 0, max_images < 0, bad grid, pointer
 * that is not device memory. */
int lh_delens_grid(const double *ax, const double *ay, const lh_grid *g, const double *sources, int nsources,
                   lh_image *images, long long max_images, long long *count);

/* ---- NEXT row f3: chi^2 of multiple-image constraints ------------------------------------------------------
 * One observed image c_k of source `source`, with its positional error sigma. */
typedef struct {
    int32_t source; /* 0 .. nsources-1 */
    int32_t _pad;
    double x, y;    /* observed position c_k */
    double sigma;   /* > 0 */
} lh_constraint;

/* chi^2 = sum_k |c_k - x_k|^2 / sigma_k^2 (eq. 6) through the four stages of PAPER.md:192-194, all on
 * the device: (1) deflection on the grid; (2) every constraint unlensed at its own position, beta_k = c_k -
 * alpha(c_k), source i = barycentre of its beta_k (Fig. 3); (3) predicted images of the sources by delensing the
 * grid (lh_delens_grid); (4) x_k = the predicted image of c_k's source closest to c_k, summed in index order.
 * A constraint whose source has no predicted image on the grid contributes +inf; a source without constraints is
 * ignored (readings R23).
 *   constraints  HOST [nconstraints], read during the call
 *   chi2         DEVICE double[1]
 *   predicted    DEVICE [nconstraints][2] or NULL: the x_k (NaN where there is none)
 *   sources      DEVICE [nsources][2] or NULL: the barycentres (NaN for a source without constraints)
 *   nimages      DEVICE long long[1] or NULL: predicted images found.  The library holds up to
 *                64*nconstraints + 4096 of them; beyond that chi2 is NaN.
 * Asynchronous on the set stream.  LH_EINVAL: as lh_grid_gradient, plus source index outside [0, nsources),
 * sigma <= 0 or non-finite constraint. */
int lh_chi2(const lh_lens *lenses, int nlens, const lh_grid *g, const lh_constraint *constraints, int nconstraints,
            int nsources, double *chi2, double *predicted, double *sources, long long *nimages);

/* Same as lh_grid_eval_batch with HOST output planes: the library allocates (and
 * caches) device planes, runs the same kernel, copies the requested planes back
 * and synchronises the stream before returning.  Large jobs are cut into up to 8
 * pieces (row slabs of one map, groups of models of a batch) so that the copy of one
 * piece overlaps the computation of the next; the results are bit-identical to the
 * device entry point's.  This is the end-to-end path a
 * caller without device buffers uses. */
int lh_grid_eval_host(const lh_lens *lenses, int nmodel, int nlens, const lh_grid *g, const lh_outputs *host_o);

/* Rows [j0, j0 + nrows) of ONE map into HOST planes of nrows*nx doubles each: the host-memory form of
 * lh_grid_eval_rows (the multi-GPU row-slab primitive; "the grid is split among the GPUs"), pipelined
 * like lh_grid_eval_host.  Pixel coordinates are those of the full grid, so the slabs of several devices stacked are
 * bit-identical to the single-device map.  Synchronises the set stream.  Errors as lh_grid_eval_host, plus
 * LH_EINVAL for a slab outside the grid. */
int lh_grid_eval_rows_host(const lh_lens *lenses, int nlens, const lh_grid *g, int j0, int nrows,
                           const lh_outputs *host_outputs);

/* CUDA stream (a cudaStream_t / CUstream cast to void*) used by later calls from
 * this host thread; NULL = legacy default stream.  Always returns LH_OK. */
int lh_set_stream(void *cuda_stream);

/* Message for the last non-zero return on this host thread ("" if none). */
const char *lh_last_error(void);

/* Step a1 on its own (host only, no CUDA call): validate `n` lenses of one model and
 * write the per-lens constant table the kernels consume -- n records of
 * LH_PACK_DOUBLES doubles, sorted by evaluation class (stable inside a class) -- into
 * host memory `table`, and the class boundaries into class_begin[0..LH_PACK_CLASSES]
 * (class k = records [class_begin[k], class_begin[k+1])).  `table` may be NULL to
 * validate only.  Returns LH_OK or LH_EINVAL (rules as lh_grid_gradient). */
#define LH_PACK_DOUBLES 24
#define LH_PACK_CLASSES 4
int lh_pack_model(const lh_lens *lenses, int n, double *table, int32_t *class_begin);

/* ---- several GPUs, one process each: writing a row slab straight into the owner's map ----
 * The output planes of lh_grid_eval_rows are plain device pointers, so a rank may hand it the address of ITS rows
 * inside a map that lives on ANOTHER device: the kernel's epilogue stores then travel over NVLink (peer access) while
 * the rest of the grid is still computing, and the one map is assembled with no gather and no second pass
 * (PAPER.md:194 "the grid is split among the GPUs"; pixels are independent, :175).  Across processes the owner's buffer
 * is reached through CUDA IPC; these three calls are thin wrappers of cudaIpcGetMemHandle / cudaIpcOpenMemHandle /
 * cudaIpcCloseMemHandle that also deal with a buffer sitting inside a larger allocation (a caching allocator's).
 *   lh_ipc_export  `dev_ptr`: device memory of THIS process.  Writes the 64-byte handle of the allocation that holds
 *                  it and the byte offset of `dev_ptr` inside that allocation.
 *   lh_ipc_open    maps the exporter's allocation into this process (another process than the exporter) and returns
 *                  the address that corresponds to the exported `dev_ptr`.  The exporter's device must be the current
 *                  one or peer-accessible from it.
 *   lh_ipc_close   unmaps it (the pointer lh_ipc_open returned).
 * Ordering is the caller's: the owner may read its map once every writer's stream has been synchronised (e.g. a
 * barrier after torch.cuda.synchronize()).  LH_EINVAL: NULL argument, unknown pointer; LH_ECUDA: a CUDA call failed. */
#define LH_IPC_HANDLE_BYTES 64
int lh_ipc_export(const void *dev_ptr, unsigned char handle[LH_IPC_HANDLE_BYTES], unsigned long long *offset);
int lh_ipc_open(const unsigned char handle[LH_IPC_HANDLE_BYTES], unsigned long long offset, void **dev_ptr);
int lh_ipc_close(void *dev_ptr);

/* "lh <major>.<minor> sm_100a" */
const char *lh_version(void);

/* Diagnostics (launch counter, FP64 peak probe, host evaluation of the kernel's primitives, source hash, and the
 * checking build's address-range calls) are declared in lh_diag.h: they serve bench.py and the tests, not the method. */

#ifdef __cplusplus
}
#endif
#endif /* LH_H_ */

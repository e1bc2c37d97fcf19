// lh_delens.cu -- NEXT row f1: source-plane map and brute-force delensing (R22).
//
//   beta = theta - alpha(theta)                                         PAPER.md:39 (eq. 1)
//   "unlens a image-plane grid unto the source-plane and check each quadrant for the presence of the
//    source (see Fig.4)"                                                PAPER.md:87-91 (sec. 2.3)
//   "searching for the images by delensing and checking the grid for sources ... Each image found is
//    stored ... divergent execution path"                               PAPER.md:194 (sec. 4.2)
//
// One thread owns one grid cell (two triangles, cut along V10-V01); a CTA owns a tile of 32 x 8 cells.
// The sources of a launch travel in the kernel parameters.  A tile first keeps the sources that fall in
// the bounding box of ALL its cells' source-plane corners (shared memory list, typically empty); a cell
// then rejects those against the box of its own four corners (that box contains the boxes of both
// triangles, so nothing the definition accepts is lost) and only then runs, per triangle, the
// definition of R22: closed bounding box of the three vertices AND the barycentric test.  The test arithmetic is written with the round-to-nearest intrinsics, i.e. WITHOUT FMA
// contraction: it takes an integer decision (inside / outside) and must take it in exactly the
// arithmetic the definition states, so that a triangle id never depends on the compiler.
// Found images are appended through one atomic counter (order is not defined).
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/lh.h"
#include "lh_kernels.h"

namespace lh {

constexpr int DELENS_SOURCES = 1024;  // sources per launch (16 KB of the 32 KB parameter space)
constexpr int DELENS_THREADS = 256;

struct DelensParams {
    const double *ax, *ay;
    lh_image *images;
    unsigned long long *count;
    long long max_images;
    double x0, y0, dx;
    int nx, ny;
    int source0, nsources;  // global index of src[0]; sources in this launch
    const double *dsrc;     // DEV_SRC variant: DEVICE [nsources][2] (f3: sources computed on the device); else nullptr
    double src[DELENS_SOURCES][2];
};
static_assert(sizeof(DelensParams) <= 32764, "kernel parameter space");

__device__ __forceinline__ double cross_rn(double ax, double ay, double bx, double by) {
    return __dsub_rn(__dmul_rn(ax, by), __dmul_rn(ay, bx));
}

__device__ __forceinline__ void test_triangle(const DelensParams &P, int s, double sx, double sy, const double (&T)[4][2],
                                              const double (&B)[4][2], int a, int b, int c, long long tri) {
    // R22: inside = inside the closed bounding box of the triangle's three vertices AND the barycentric test
    if (sx < fmin(fmin(B[a][0], B[b][0]), B[c][0]) || sx > fmax(fmax(B[a][0], B[b][0]), B[c][0]) ||
        sy < fmin(fmin(B[a][1], B[b][1]), B[c][1]) || sy > fmax(fmax(B[a][1], B[b][1]), B[c][1]))
        return;
    const double e1x = __dsub_rn(B[b][0], B[a][0]), e1y = __dsub_rn(B[b][1], B[a][1]);
    const double e2x = __dsub_rn(B[c][0], B[a][0]), e2y = __dsub_rn(B[c][1], B[a][1]);
    const double px = __dsub_rn(sx, B[a][0]), py = __dsub_rn(sy, B[a][1]);
    const double d = cross_rn(e1x, e1y, e2x, e2y);
    if (d == 0.0) return;
    const double u = __ddiv_rn(cross_rn(px, py, e2x, e2y), d);
    const double v = __ddiv_rn(cross_rn(e1x, e1y, px, py), d);
    if (!(u >= 0.0 && v >= 0.0 && __dadd_rn(u, v) <= 1.0)) return;
    const unsigned long long k = atomicAdd(P.count, 1ULL);
    if (k >= (unsigned long long)P.max_images) return;
    lh_image im;
    im.source = P.source0 + s;
    im._pad = 0;
    im.triangle = tri;
    im.x = __dadd_rn(__dadd_rn(T[a][0], __dmul_rn(u, __dsub_rn(T[b][0], T[a][0]))), __dmul_rn(v, __dsub_rn(T[c][0], T[a][0])));
    im.y = __dadd_rn(__dadd_rn(T[a][1], __dmul_rn(u, __dsub_rn(T[b][1], T[a][1]))), __dmul_rn(v, __dsub_rn(T[c][1], T[a][1])));
    P.images[k] = im;
}

// A CTA owns a tile of TILE_CW x TILE_CH cells (one warp per cell row, coalesced vertex loads) and walks the tiles
// of the grid persistently.  Per tile: (1) every thread maps the four corners of its cell to the source plane and
// takes their bounding box; (2) the boxes are reduced to the box of the TILE; (3) the threads scan the source list
// together and keep, in shared memory, the few sources inside the tile's box; (4) every thread runs the R22 test of
// its cell against those survivors only.  Steps (2)-(3) are a superset filter (a source outside the tile's box is
// outside the box of each of its cells), so the images found are exactly those of the plain cell x source loop.
constexpr int TILE_CW = 32, TILE_CH = DELENS_THREADS / 32;

__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

template <bool DEV_SRC>
__global__ void __launch_bounds__(DELENS_THREADS) delens_kernel(const __grid_constant__ DelensParams P) {
    __shared__ double s_part[TILE_CH][4];     // per-warp box: lox, hix, loy, hiy
    __shared__ double s_box[4];               // box of the tile
    __shared__ int s_n;                       // survivors of the current pass
    __shared__ int s_idx[DELENS_SOURCES];     // their indices into the launch's source list
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ncx = P.nx - 1, ncy = P.ny - 1;
    const int tiles_x = (ncx + TILE_CW - 1) / TILE_CW, tiles_y = (ncy + TILE_CH - 1) / TILE_CH;
    const long long ntiles = (long long)tiles_x * tiles_y;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int ty = (int)(tile / tiles_x), tx = (int)(tile - (long long)ty * tiles_x);
        const int i = tx * TILE_CW + lane, j = ty * TILE_CH + warp;
        const bool valid = i < ncx && j < ncy;
        const long long cell = (long long)j * ncx + i;
        double T[4][2], B[4][2];  // corners 00, 10, 01, 11 in the image plane and in the source plane
        double lox = INFINITY, hix = -INFINITY, loy = INFINITY, hiy = -INFINITY;
        if (valid) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int ii = i + (c & 1), jj = j + (c >> 1);
                const size_t p = (size_t)jj * P.nx + ii;
                T[c][0] = __dadd_rn(P.x0, __dmul_rn((double)ii, P.dx));
                T[c][1] = __dadd_rn(P.y0, __dmul_rn((double)jj, P.dx));
                B[c][0] = __dsub_rn(T[c][0], __ldg(P.ax + p));
                B[c][1] = __dsub_rn(T[c][1], __ldg(P.ay + p));
                lox = fmin(lox, B[c][0]); hix = fmax(hix, B[c][0]);
                loy = fmin(loy, B[c][1]); hiy = fmax(hiy, B[c][1]);
            }
        }
        // (2) box of the tile.  fmin / fmax drop NaN corners (a NaN deflection never yields an image: every
        // comparison of the cell's own test below is false for it)
        {
            const double a = warp_min(lox), b = warp_max(hix), c = warp_min(loy), d = warp_max(hiy);
            if (lane == 0) { s_part[warp][0] = a; s_part[warp][1] = b; s_part[warp][2] = c; s_part[warp][3] = d; }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double a = s_part[0][0], b = s_part[0][1], c = s_part[0][2], d = s_part[0][3];
            for (int w = 1; w < TILE_CH; ++w) {
                a = fmin(a, s_part[w][0]); b = fmax(b, s_part[w][1]);
                c = fmin(c, s_part[w][2]); d = fmax(d, s_part[w][3]);
            }
            s_box[0] = a; s_box[1] = b; s_box[2] = c; s_box[3] = d;
        }
        // DEV_SRC: the device list may be longer than one pass holds
        for (int s0 = 0; s0 < P.nsources; s0 += DELENS_SOURCES) {
            const int ns = P.nsources - s0 < DELENS_SOURCES ? P.nsources - s0 : DELENS_SOURCES;
            if (threadIdx.x == 0) s_n = 0;
            __syncthreads();
            // (3) sources inside the tile's box (NaN sources -- chi^2 sources without constraints -- fail the test)
            const double tlox = s_box[0], thix = s_box[1], tloy = s_box[2], thiy = s_box[3];
            for (int s = threadIdx.x; s < ns; s += DELENS_THREADS) {
                const double sx = DEV_SRC ? __ldg(P.dsrc + 2 * (s0 + s)) : P.src[s][0];
                const double sy = DEV_SRC ? __ldg(P.dsrc + 2 * (s0 + s) + 1) : P.src[s][1];
                if (sx >= tlox && sx <= thix && sy >= tloy && sy <= thiy) s_idx[atomicAdd(&s_n, 1)] = s;
            }
            __syncthreads();
            // (4) the cell's own test on the survivors
            const int n = s_n;
            if (valid) {
                for (int q = 0; q < n; ++q) {
                    const int s = s_idx[q];
                    const double sx = DEV_SRC ? __ldg(P.dsrc + 2 * (s0 + s)) : P.src[s][0];
                    const double sy = DEV_SRC ? __ldg(P.dsrc + 2 * (s0 + s) + 1) : P.src[s][1];
                    // outside the box of the four corners = outside the box of either triangle (R22): reject
                    if (sx < lox || sx > hix || sy < loy || sy > hiy) continue;
                    test_triangle(P, s0 + s, sx, sy, T, B, 0, 1, 2, 2 * cell);
                    test_triangle(P, s0 + s, sx, sy, T, B, 3, 2, 1, 2 * cell + 1);
                }
            }
            __syncthreads();  // s_n / s_idx / s_box are rewritten by the next pass or tile
        }
    }
}

__global__ void __launch_bounds__(256) source_plane_kernel(const double *__restrict__ ax, const double *__restrict__ ay,
                                                           double x0, double y0, double dx, int nx, int ny,
                                                           double *__restrict__ bx, double *__restrict__ by) {
    const long long n = (long long)nx * ny;
    for (long long p = (long long)blockIdx.x * 256 + threadIdx.x; p < n; p += (long long)gridDim.x * 256) {
        const int j = (int)(p / nx), i = (int)(p - (long long)j * nx);
        if (bx) bx[p] = __dsub_rn(__dadd_rn(x0, __dmul_rn((double)i, dx)), ax[p]);
        if (by) by[p] = __dsub_rn(__dadd_rn(y0, __dmul_rn((double)j, dx)), ay[p]);
    }
}

cudaError_t launch_source_plane(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                                double *bx, double *by, int sms, cudaStream_t st) {
    const long long n = (long long)nx * ny;
    long long blocks = (n + 255) / 256;
    if (blocks > (long long)sms * 16) blocks = (long long)sms * 16;
    source_plane_kernel<<<(unsigned)blocks, 256, 0, st>>>(ax, ay, x0, y0, dx, nx, ny, bx, by);
    return cudaGetLastError();
}

// sources: HOST [ns][2].  One launch per DELENS_SOURCES sources; `count` must be zero on entry.
cudaError_t launch_delens(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                          const double *sources, int ns, lh_image *images, long long max_images,
                          unsigned long long *count, int sms, cudaStream_t st, long long *launches) {
    thread_local DelensParams P;
    P.ax = ax; P.ay = ay; P.images = images; P.count = count; P.max_images = max_images;
    P.x0 = x0; P.y0 = y0; P.dx = dx; P.nx = nx; P.ny = ny;
    const long long ncells = (long long)(nx - 1) * (ny - 1);
    if (ncells <= 0) return cudaSuccess;
    long long blocks = (long long)((nx - 1 + TILE_CW - 1) / TILE_CW) * ((ny - 1 + TILE_CH - 1) / TILE_CH);
    if (blocks > (long long)sms * 8) blocks = (long long)sms * 8;  // persistent: 8 CTAs of 256 threads per SM
    for (int s0 = 0; s0 < ns; s0 += DELENS_SOURCES) {
        const int n = ns - s0 < DELENS_SOURCES ? ns - s0 : DELENS_SOURCES;
        P.source0 = s0; P.nsources = n;
        for (int s = 0; s < n; ++s) { P.src[s][0] = sources[2 * (s0 + s)]; P.src[s][1] = sources[2 * (s0 + s) + 1]; }
        P.dsrc = nullptr;
        delens_kernel<false><<<(unsigned)blocks, DELENS_THREADS, 0, st>>>(P);
        ++*launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// sources: DEVICE [ns][2] (a NaN source matches nothing).  One launch; `count` must be zero on entry.
cudaError_t launch_delens_dev(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                              const double *dsources, int ns, lh_image *images, long long max_images,
                              unsigned long long *count, int sms, cudaStream_t st, long long *launches) {
    thread_local DelensParams P;
    P.ax = ax; P.ay = ay; P.images = images; P.count = count; P.max_images = max_images;
    P.x0 = x0; P.y0 = y0; P.dx = dx; P.nx = nx; P.ny = ny;
    P.source0 = 0; P.nsources = ns; P.dsrc = dsources;
    const long long ncells = (long long)(nx - 1) * (ny - 1);
    if (ncells <= 0 || ns <= 0) return cudaSuccess;
    long long blocks = (long long)((nx - 1 + TILE_CW - 1) / TILE_CW) * ((ny - 1 + TILE_CH - 1) / TILE_CH);
    if (blocks > (long long)sms * 8) blocks = (long long)sms * 8;
    delens_kernel<true><<<(unsigned)blocks, DELENS_THREADS, 0, st>>>(P);
    ++*launches;
    return cudaGetLastError();
}

// ---- f3: the small stages of the chi^2 pipeline (PAPER.md:76-81 eq. 6, :192-194; readings R23) -------------
__global__ void constraint_points_kernel(const lh_constraint *c, int K, double *cx, double *cy) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < K) { cx[k] = c[k].x; cy[k] = c[k].y; }
}

// stage 2: source i = barycentre of beta_k = c_k - alpha(c_k) over its constraints, summed in index order
__global__ void barycentre_kernel(const lh_constraint *c, int K, const double *ax, const double *ay, int nsources,
                                  double *src) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsources) return;
    double sx = 0.0, sy = 0.0;
    int n = 0;
    for (int k = 0; k < K; ++k) {
        if (c[k].source != i) continue;
        sx = __dadd_rn(sx, __dsub_rn(c[k].x, ax[k]));
        sy = __dadd_rn(sy, __dsub_rn(c[k].y, ay[k]));
        ++n;
    }
    src[2 * i] = n ? __ddiv_rn(sx, (double)n) : NAN;
    src[2 * i + 1] = n ? __ddiv_rn(sy, (double)n) : NAN;
}

// stage 4a: x_k = predicted image of the constraint's source closest to it; term_k = |c_k - x_k|^2 / sigma_k^2
__global__ void assign_kernel(const lh_constraint *c, int K, const lh_image *im, const unsigned long long *count,
                              long long cap, double *pred, double *term) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const long long n = *count < (unsigned long long)cap ? (long long)*count : cap;
    double best = INFINITY, bx = NAN, by = NAN;
    for (long long m = 0; m < n; ++m) {
        if (im[m].source != c[k].source) continue;
        const double ex = __dsub_rn(c[k].x, im[m].x), ey = __dsub_rn(c[k].y, im[m].y);
        const double d2 = __dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey));
        if (d2 < best) { best = d2; bx = im[m].x; by = im[m].y; }
    }
    if (pred) { pred[2 * k] = bx; pred[2 * k + 1] = by; }
    term[k] = __ddiv_rn(best, __dmul_rn(c[k].sigma, c[k].sigma));
}

// stage 4b: chi^2 = sum of the terms in index order (one thread: K is a few hundred; the order is the definition's).
// More images than the buffer holds -> NaN (the assignment above did not see them all).
__global__ void chi2_sum_kernel(const double *term, int K, const unsigned long long *count, long long cap, double *chi2,
                                long long *nimages) {
    double s = 0.0;
    for (int k = 0; k < K; ++k) s = __dadd_rn(s, term[k]);
    *chi2 = (*count > (unsigned long long)cap) ? NAN : s;
    if (nimages) *nimages = (long long)*count;
}

cudaError_t launch_constraint_points(const lh_constraint *c, int K, double *cx, double *cy, cudaStream_t st) {
    if (K > 0) constraint_points_kernel<<<(K + 127) / 128, 128, 0, st>>>(c, K, cx, cy);
    return cudaGetLastError();
}
cudaError_t launch_barycentre(const lh_constraint *c, int K, const double *ax, const double *ay, int nsources, double *src,
                              cudaStream_t st) {
    if (nsources > 0) barycentre_kernel<<<(nsources + 127) / 128, 128, 0, st>>>(c, K, ax, ay, nsources, src);
    return cudaGetLastError();
}
cudaError_t launch_assign_and_sum(const lh_constraint *c, int K, const lh_image *im, const unsigned long long *count,
                                  long long cap, double *pred, double *term, double *chi2, long long *nimages,
                                  cudaStream_t st) {
    if (K > 0) assign_kernel<<<(K + 127) / 128, 128, 0, st>>>(c, K, im, count, cap, pred, term);
    chi2_sum_kernel<<<1, 1, 0, st>>>(term, K, count, cap, chi2, nimages);
    return cudaGetLastError();
}

}  // namespace lh

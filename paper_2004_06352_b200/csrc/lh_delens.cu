// lh_delens.cu -- NEXT row f1: source-plane map and brute-force delensing (R22).
//
//   beta = theta - alpha(theta)                                         PAPER.md:39 (eq. 1)
//   "unlens a image-plane grid unto the source-plane and check each quadrant for the presence of the
//    source (see Fig.4)"                                                PAPER.md:87-91 (sec. 2.3)
//   "searching for the images by delensing and checking the grid for sources ... Each image found is
//    stored ... divergent execution path"                               PAPER.md:194 (sec. 4.2)
//
// One lane owns one grid cell (two triangles, cut along V10-V01); a warp owns a tile of 32 x 8 cells.
// The sources of a launch travel in the kernel parameters.  A tile first keeps the sources that fall in
// the bounding box of ALL its vertices' source-plane images (typically none); a cell
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

// A WARP owns a tile of TILE_CW x TILE_CH cells = (TILE_CW + 1) x (TILE_CH + 1) vertices, and there is no shared
// memory and no block barrier.  Per tile: (1) lane l loads vertex column i0 + l for the TILE_CH + 1 vertex rows (all
// loads issued before the first use: 18 coalesced 256-byte requests in flight per warp) and lanes 0..TILE_CH load the
// one extra column i0 + 32 -- every vertex is fetched and mapped to the source plane ONCE per tile; (2) each lane
// folds its vertices into a box and five shuffle steps per bound make the box of the TILE; (3) the warp scans the
// source list 32 at a time against that box (one ballot per 32 sources).  Almost every tile ends here.  (4) For a
// source that survives, every lane runs the R22 test of its cell in each of the tile's rows, reloading the four
// corners (L1 hits).  Steps (2)-(3) are a superset filter -- the tile's box contains the box of each of its cells, and
// fmin / fmax drop NaN corners, which never yield an image anyway -- so the images found are exactly those of the
// plain cell x source loop, and the deciding arithmetic of step (4) is the definition's, untouched.
// Round 2's kernel did the same filter per CTA with three block barriers and a one-thread reduction per tile and
// fetched every vertex four times: 0.543 ms on 4096^2 x 80 sources, latency-bound at 0.08 of HBM.
constexpr int TILE_CW = 32, TILE_CH = 8;
constexpr int DELENS_WARPS = DELENS_THREADS / 32;
#ifndef LH_DELENS_MINB
#define LH_DELENS_MINB 4  // CTAs per SM the registers are held to (64); the first, shuffle-based version of this kernel measured 0.135 ms at 4, 0.141 at 3, 0.158 at 2
#endif

// The filter of steps (2)-(3) works on a monotone 32-bit KEY of a double instead of the double itself: the high word
// with the sign folded in, so that x <= y implies key(x) <= key(y) (unsigned; equal keys for doubles that differ in
// the low word only).  lo <= s <= hi therefore implies key(lo) <= key(s) <= key(hi): testing keys can only let MORE
// sources through than testing doubles, never fewer, which is all a superset filter needs -- and keys take one
// integer min / max per vertex and one hardware warp reduction (redux.sync) per bound, where doubles took a
// multi-instruction fmin / fmax and ten shuffles (ncu on the first version of this kernel: 942 instructions per tile,
// short-scoreboard stalls from the 80 shuffles on top).  NaN and infinite vertices give extreme keys = a wider box.
__device__ __forceinline__ unsigned key32(double x) {
    const int h = __double2hiint(x);
    return (unsigned)h ^ ((unsigned)(h >> 31) | 0x80000000u);
}

// step (4) for one cell and one source: corners 00, 10, 01, 11 in the image plane and in the source plane, the box
// of the four corners (it contains the boxes of both triangles, so nothing the definition accepts is lost), then the
// definition per triangle.  Rare; kept out of line so that the streaming loop stays small.
__device__ __noinline__ void cell_test(const DelensParams &P, int s, double sx, double sy, int i, int j) {
    const long long cell = (long long)j * (P.nx - 1) + i;
    double T[4][2], B[4][2];
    double lox = INFINITY, hix = -INFINITY, loy = INFINITY, hiy = -INFINITY;
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
    if (sx < lox || sx > hix || sy < loy || sy > hiy) return;
    test_triangle(P, s, sx, sy, T, B, 0, 1, 2, 2 * cell);
    test_triangle(P, s, sx, sy, T, B, 3, 2, 1, 2 * cell + 1);
}

template <bool DEV_SRC>
__global__ void __launch_bounds__(DELENS_THREADS, LH_DELENS_MINB) delens_kernel(const __grid_constant__ DelensParams P) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ncx = P.nx - 1, ncy = P.ny - 1;
    const int tiles_x = (ncx + TILE_CW - 1) / TILE_CW, tiles_y = (ncy + TILE_CH - 1) / TILE_CH;
    const long long ntiles = (long long)tiles_x * tiles_y;
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    for (long long tile = (long long)blockIdx.x * DELENS_WARPS + warp; tile < ntiles; tile += (long long)gridDim.x * DELENS_WARPS) {
        const int ty = (int)(tile / tiles_x), tx = (int)(tile - (long long)ty * tiles_x);
        const int i0 = tx * TILE_CW, j0 = ty * TILE_CH;
        // the sources of a scan step are requested one step ahead, the first before the vertices (ncu: 28 % of the samples
        // of the version without this sat on the wait for the indexed constant-bank load; ptxas still places the first
        // request behind the vertex loads, so the measured gain is nil -- 119 vs 121 us -- and the wait remains the top stall)
        double sx = qnan, sy = qnan;
        if (lane < P.nsources) {
            sx = DEV_SRC ? __ldg(P.dsrc + 2 * lane) : P.src[lane][0];
            sy = DEV_SRC ? __ldg(P.dsrc + 2 * lane + 1) : P.src[lane][1];
        }
        // (1) this lane's vertex column, rows j0 .. j0 + TILE_CH; an index outside the grid is clamped to the last vertex
        // of the grid in that direction (a vertex of this tile: counting it twice leaves the box unchanged)
        const int vi = i0 + lane, ci = vi < P.nx ? vi : P.nx - 1;
        double vx[TILE_CH + 1], vy[TILE_CH + 1];
#pragma unroll
        for (int r = 0; r <= TILE_CH; ++r) {
            const int cj = j0 + r < P.ny ? j0 + r : P.ny - 1;
            const size_t p = (size_t)cj * P.nx + ci;
            vx[r] = __ldg(P.ax + p);
            vy[r] = __ldg(P.ay + p);
        }
        // the extra column i0 + TILE_CW: lane r takes its row r (the other lanes repeat row TILE_CH)
        const int ei = i0 + TILE_CW < P.nx ? i0 + TILE_CW : P.nx - 1;
        const int er = lane <= TILE_CH ? lane : TILE_CH, ej = j0 + er < P.ny ? j0 + er : P.ny - 1;
        const double ex = __ldg(P.ax + (size_t)ej * P.nx + ei);
        const double ey = __ldg(P.ay + (size_t)ej * P.nx + ei);
        // (2) box of the tile's vertices in the source plane, in keys: beta = theta - alpha, theta as step (4) forms it
        const double thx = __dadd_rn(P.x0, __dmul_rn((double)ci, P.dx));
        unsigned lox = 0xffffffffu, hix = 0u, loy = 0xffffffffu, hiy = 0u;
#pragma unroll
        for (int r = 0; r <= TILE_CH; ++r) {
            const int cj = j0 + r < P.ny ? j0 + r : P.ny - 1;
            const unsigned kx = key32(__dsub_rn(thx, vx[r]));
            const unsigned ky = key32(__dsub_rn(__dadd_rn(P.y0, __dmul_rn((double)cj, P.dx)), vy[r]));
            lox = min(lox, kx); hix = max(hix, kx);
            loy = min(loy, ky); hiy = max(hiy, ky);
        }
        {
            const unsigned kx = key32(__dsub_rn(__dadd_rn(P.x0, __dmul_rn((double)ei, P.dx)), ex));
            const unsigned ky = key32(__dsub_rn(__dadd_rn(P.y0, __dmul_rn((double)ej, P.dx)), ey));
            lox = min(lox, kx); hix = max(hix, kx);
            loy = min(loy, ky); hiy = max(hiy, ky);
        }
        const unsigned tlox = __reduce_min_sync(0xffffffffu, lox), thix = __reduce_max_sync(0xffffffffu, hix);
        const unsigned tloy = __reduce_min_sync(0xffffffffu, loy), thiy = __reduce_max_sync(0xffffffffu, hiy);
        // (3) the source list, 32 sources per step.  (A NaN source -- a chi^2 source without constraints -- has an
        // extreme key and normally fails here; where it does not, every comparison of step (4) is false for it.)
        for (int s0 = 0; s0 < P.nsources; s0 += 32) {
            const int s = s0 + lane, sn = s + 32;
            double nsx = qnan, nsy = qnan;  // the next step's sources, one step ahead
            if (sn < P.nsources) {
                nsx = DEV_SRC ? __ldg(P.dsrc + 2 * sn) : P.src[sn][0];
                nsy = DEV_SRC ? __ldg(P.dsrc + 2 * sn + 1) : P.src[sn][1];
            }
            const unsigned ksx = key32(sx), ksy = key32(sy);
            unsigned m = __ballot_sync(0xffffffffu, s < P.nsources && ksx >= tlox && ksx <= thix && ksy >= tloy && ksy <= thiy);
            // (4) rare: the cells of the tile against each survivor
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                const double qx = __shfl_sync(0xffffffffu, sx, b), qy = __shfl_sync(0xffffffffu, sy, b);
#pragma unroll 1
                for (int r = 0; r < TILE_CH; ++r)
                    if (vi < ncx && j0 + r < ncy) cell_test(P, s0 + b, qx, qy, vi, j0 + r);
            }
            sx = nsx; sy = nsy;
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

// One warp per tile, DELENS_WARPS tiles per CTA; beyond 64 CTAs per SM the warps walk the tiles grid-stride.
static long long delens_blocks(int nx, int ny, int sms) {
    const long long tiles = (long long)((nx - 1 + TILE_CW - 1) / TILE_CW) * ((ny - 1 + TILE_CH - 1) / TILE_CH);
    long long blocks = (tiles + DELENS_WARPS - 1) / DELENS_WARPS;
    const long long cap = (long long)(sms > 0 ? sms : 148) * 64;
    return blocks > cap ? cap : (blocks < 1 ? 1 : blocks);
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
    long long blocks = delens_blocks(nx, ny, sms);
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
    long long blocks = delens_blocks(nx, ny, sms);
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

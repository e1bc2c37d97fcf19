/*
 * lens_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded, double-precision CPU statement of what the
 * lens-map hot path computes.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code, header, table or constant with the CUDA path under
 * paper_2004_06352_b200/csrc (it even declares its own lens record).
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared lens_oracle.c -lm
 *        (no FMA contraction, so results do not depend on the host ISA).
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, arXiv 2004.06352):
 *   - alpha = grad psi, lens equation            PAPER.md:39-53  (eq. 1-2)
 *   - A^-1 = delta_ij - d_ij psi, kappa, gamma   PAPER.md:57     (eq. 4)
 *   - mu = 1/det A^-1                            PAPER.md:64     (eq. 5)
 *   - kappa/gamma/mu maps from 2nd derivatives   PAPER.md:105-110 (eq. 7-9)
 *   - "at each grid-point the second-order derivative contribution of each
 *      cluster member is added up"               PAPER.md:112    (sec. 2.4)
 *   - grad phi = sum_h grad phi_h                PAPER.md:183    (eq. 10)
 * The paper never prints the potentials (PAPER.md:70 only names the parameter
 * kinds and cites ref [6]); the per-lens closed forms are the
 * reading fixed in SURVEY.md sec. 8(c) / Appendix A.1-A.3 and DESIGN.md sec. 3:
 * a PIEMD of core r has convergence kappa = 1/(2 sqrt(r^2 + rho^2)),
 * rho^2 = x'^2/(1+eps)^2 + y'^2/(1-eps)^2; NSIE = b0*PIEMD(rcore);
 * dPIE = b0*rcut/(rcut-rcore)*(PIEMD(rcore) - PIEMD(rcut)); SIS = circular,
 * r = 0.  Garbled equations are read as DESIGN.md sec. 3 lists (eq. 8: sum the
 * Hessian first, gamma1 = (a11-a22)/2, gamma2 = a12; eq. 9: minus sign).
 *
 * The dPIE is written in its straightforward two-term form (core term minus
 * cut term, libm atan/atanh/sqrt, explicit rotation matrices) -- deliberately
 * NOT the merged / rotation-free forms the GPU uses.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): Poisson integral of kappa
 * by quadrature, SURVEY Appendix B 40-digit worked example, circular dPIE and
 * SIS closed forms, linearity, finite-difference Hessian, epilogue identities,
 * rotation covariance, limits between types, far-field mass, mpmath
 * complex-log brute force.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

enum { ORC_DPIE = 0, ORC_NSIE = 1, ORC_SIS = 2 };

/* own declaration of the 64-byte boundary record (same bytes as lh_lens) */
typedef struct {
    int32_t type;
    int32_t pad_;
    double x, y;        /* centre [arcsec] */
    double ellipticity; /* e-hat = (A^2-B^2)/(A^2+B^2) of the isodensities */
    double theta;       /* major axis, CCW from +x [rad] */
    double rcore, rcut; /* [arcsec] */
    double b0;          /* [arcsec] */
} orc_lens;

/* first and second derivatives of one potential: (ax, ay, a11, a12, a22) */
typedef struct {
    double ax, ay, a11, a12, a22;
} orc_deriv;

/* Reading 8c-2: eps = e-hat / (1 + sqrt(1 - e-hat^2)) */
double orc_eps_from_ehat(double ehat) { return ehat / (1.0 + sqrt(1.0 - ehat * ehat)); }

/*
 * PIEMD kernel with core r and unit b0 in the LENS frame (Appendix A.1):
 *   Jx = o/(2 sqrt(eps)) * atan ( 2 sqrt(eps) x' / (o w + (1+eps)^2 r) )
 *   Jy = o/(2 sqrt(eps)) * atanh( 2 sqrt(eps) y' / (o w + (1-eps)^2 r) )
 *   D  = 2(1+eps^2) r^2 + 2 o r w + x'^2 + y'^2
 *   hxx = ((1-eps)^2 r^2 + o r w + y'^2)/(w D)
 *   hyy = ((1+eps)^2 r^2 + o r w + x'^2)/(w D)
 *   hxy = -x' y'/(w D)
 * with o = 1 - eps^2, w = sqrt(r^2 + rho^2).  eps -> 0 (A.2): atan(u)/u -> 1.
 */
static void piemd_kernel(double xp, double yp, double eps, double r, double *jx, double *jy, double *hxx,
                         double *hxy, double *hyy) {
    const double o = 1.0 - eps * eps;
    const double p = (1.0 + eps) * (1.0 + eps);
    const double m = (1.0 - eps) * (1.0 - eps);
    const double rho2 = xp * xp / p + yp * yp / m;
    const double w = sqrt(r * r + rho2);
    const double se2 = 2.0 * sqrt(eps);

    const double X = xp / (o * w + p * r); /* atan argument / (2 sqrt eps) */
    const double Y = yp / (o * w + m * r); /* atanh argument / (2 sqrt eps) */
    const double ux = se2 * X, uy = se2 * Y;
    /* o/(2 sqrt eps) * atan(ux) == o * X * (atan(ux)/ux); the ratio is 1 at ux = 0 */
    const double atanc = (ux != 0.0) ? atan(ux) / ux : 1.0;
    const double atanhc = (uy != 0.0) ? atanh(uy) / uy : 1.0;
    *jx = o * X * atanc;
    *jy = o * Y * atanhc;

    const double D = 2.0 * (1.0 + eps * eps) * r * r + 2.0 * o * r * w + xp * xp + yp * yp;
    const double wD = w * D;
    *hxx = (m * r * r + o * r * w + yp * yp) / wD;
    *hyy = (p * r * r + o * r * w + xp * xp) / wD;
    *hxy = -xp * yp / wD;
}

/* One potential at one point.  Types and rotation: Appendix A.3, readings 8c-1,3,11,19. */
void orc_lens_deriv(const orc_lens *L, double X, double Y, orc_deriv *out) {
    const double dx = X - L->x, dy = Y - L->y;
    out->ax = out->ay = out->a11 = out->a12 = out->a22 = 0.0;

    if (L->type == ORC_SIS) {
        /* alpha = b0 (dx,dy)/R ; H = b0/R^3 [[dy^2, -dx dy],[-dx dy, dx^2]] ; zero at R = 0 */
        const double R2 = dx * dx + dy * dy;
        if (R2 == 0.0) return;
        const double R = sqrt(R2);
        out->ax = L->b0 * dx / R;
        out->ay = L->b0 * dy / R;
        const double R3 = R2 * R;
        out->a11 = L->b0 * dy * dy / R3;
        out->a12 = -L->b0 * dx * dy / R3;
        out->a22 = L->b0 * dx * dx / R3;
        return;
    }

    const double c = cos(L->theta), s = sin(L->theta);
    const double xp = c * dx + s * dy;  /* lens frame: x' along the major axis */
    const double yp = -s * dx + c * dy;
    const double eps = orc_eps_from_ehat(L->ellipticity);

    double jx, jy, hxx, hxy, hyy; /* lens-frame alpha' and H' */
    if (L->type == ORC_NSIE) {
        piemd_kernel(xp, yp, eps, L->rcore, &jx, &jy, &hxx, &hxy, &hyy);
        jx *= L->b0; jy *= L->b0; hxx *= L->b0; hxy *= L->b0; hyy *= L->b0;
    } else { /* ORC_DPIE: core term minus cut term */
        double jxc, jyc, hxxc, hxyc, hyyc, jxt, jyt, hxxt, hxyt, hyyt;
        piemd_kernel(xp, yp, eps, L->rcore, &jxc, &jyc, &hxxc, &hxyc, &hyyc);
        piemd_kernel(xp, yp, eps, L->rcut, &jxt, &jyt, &hxxt, &hxyt, &hyyt);
        const double T = L->b0 * L->rcut / (L->rcut - L->rcore);
        jx = T * (jxc - jxt);
        jy = T * (jyc - jyt);
        hxx = T * (hxxc - hxxt);
        hxy = T * (hxyc - hxyt);
        hyy = T * (hyyc - hyyt);
    }
    /* back-rotation alpha = R(theta) alpha', H = R H' R^T */
    out->ax = c * jx - s * jy;
    out->ay = s * jx + c * jy;
    out->a11 = c * c * hxx - 2.0 * c * s * hxy + s * s * hyy;
    out->a22 = s * s * hxx + 2.0 * c * s * hxy + c * c * hyy;
    out->a12 = c * s * (hxx - hyy) + (c * c - s * s) * hxy;
}

/* Superposition in lens-index order (eq. 10; sec. 2.4). */
void orc_point(const orc_lens *lenses, int nlens, double X, double Y, orc_deriv *sum) {
    orc_deriv acc = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (int l = 0; l < nlens; ++l) {
        orc_deriv d;
        orc_lens_deriv(&lenses[l], X, Y, &d);
        acc.ax += d.ax;
        acc.ay += d.ay;
        acc.a11 += d.a11;
        acc.a12 += d.a12;
        acc.a22 += d.a22;
    }
    *sum = acc;
}

/* Epilogue (eq. 4, 5, 7-9 as read in DESIGN.md sec. 3; Appendix A.6). */
void orc_epilogue(double a11, double a12, double a22, double *kappa, double *gamma1, double *gamma2, double *mu) {
    const double k = 0.5 * (a11 + a22);
    const double g1 = 0.5 * (a11 - a22);
    const double g2 = a12;
    const double det = (1.0 - k) * (1.0 - k) - g1 * g1 - g2 * g2;
    *kappa = k;
    *gamma1 = g1;
    *gamma2 = g2;
    *mu = 1.0 / det; /* IEEE: +-inf on a critical line */
}

/* the nine output planes; a NULL plane is not written */
typedef struct {
    double *ax, *ay, *a11, *a12, *a22, *kappa, *gamma1, *gamma2, *mu;
} orc_planes;

static void store(const orc_planes *o, size_t idx, const orc_deriv *d) {
    double k, g1, g2, mu;
    orc_epilogue(d->a11, d->a12, d->a22, &k, &g1, &g2, &mu);
    if (o->ax) o->ax[idx] = d->ax;
    if (o->ay) o->ay[idx] = d->ay;
    if (o->a11) o->a11[idx] = d->a11;
    if (o->a12) o->a12[idx] = d->a12;
    if (o->a22) o->a22[idx] = d->a22;
    if (o->kappa) o->kappa[idx] = k;
    if (o->gamma1) o->gamma1[idx] = g1;
    if (o->gamma2) o->gamma2[idx] = g2;
    if (o->mu) o->mu[idx] = mu;
}

/* arbitrary points: out planes hold npts values each */
void orc_points(const orc_lens *lenses, int nlens, const double *xs, const double *ys, size_t npts,
                const orc_planes *o) {
    for (size_t k = 0; k < npts; ++k) {
        orc_deriv d;
        orc_point(lenses, nlens, xs[k], ys[k], &d);
        store(o, k, &d);
    }
}

/*
 * Rows [j0, j1) of the regular grid: pixel (i, j) at (x0 + i*dx, y0 + j*dx),
 * plane index j*nx + i ("rectangular grid ... each grid cell the
 * size of a pixel"; reading 8c-10).  Planes are FULL ny*nx maps; only the row
 * range is written, so disjoint ranges can run on different host threads.
 */
void orc_grid_rows(const orc_lens *lenses, int nlens, double x0, double y0, double dx, int nx, int ny, int j0,
                   int j1, const orc_planes *o) {
    (void)ny;
    for (int j = j0; j < j1; ++j) {
        const double Y = y0 + (double)j * dx;
        for (int i = 0; i < nx; ++i) {
            const double X = x0 + (double)i * dx;
            orc_deriv d;
            orc_point(lenses, nlens, X, Y, &d);
            store(o, (size_t)j * (size_t)nx + (size_t)i, &d);
        }
    }
}

/*
 * ---- NEXT row f1: source plane and brute-force delensing -----------------------------------
 * Lens equation beta = theta - alpha(theta)                       PAPER.md:39 (eq. 1)
 * "the 'brute force' approach is to unlens a image-plane grid unto the source-plane and check each
 * quadrant for the presence of the source (see Fig.4)"            PAPER.md:87-91 (sec. 2.3)
 * "searching for the images by delensing and checking the grid for sources ... Each image found is
 * stored"                                                         PAPER.md:194 (sec. 4.2, stage 3)
 * The paper gives no triangulation, inside rule or image position; readings R22:
 *   - vertices are the grid pixels; cell (i, j), 0 <= i < nx-1, 0 <= j < ny-1, has the corners
 *     V00 = (i, j), V10 = (i+1, j), V01 = (i, j+1), V11 = (i+1, j+1) and is cut along V10-V01 into
 *     triangle 0 = (V00, V10, V01) and triangle 1 = (V11, V01, V10); triangle id = 2*(j*(nx-1)+i)+t;
 *   - with A, B, C the triangle's vertices mapped to the source plane and S the source,
 *     d = (B-A) x (C-A), u = (S-A) x (C-A) / d, v = (B-A) x (S-A) / d; the source is inside iff
 *     d != 0, u >= 0, v >= 0 and u + v <= 1 (closed triangle: a source exactly on a shared edge is
 *     reported by both neighbours);
 *   - the image is the same barycentric combination of the image-plane vertices:
 *     theta = tA + u (tB - tA) + v (tC - tA).
 * Images are emitted in triangle order, sources in index order inside a triangle.
 */
typedef struct {
    int32_t source;   /* index into the source list */
    int32_t pad_;
    int64_t triangle; /* 2*(j*(nx-1)+i) + t */
    double x, y;      /* image position in the image plane */
} orc_image;

void orc_source_plane(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                      double *bx, double *by) {
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const size_t p = (size_t)j * (size_t)nx + (size_t)i;
            bx[p] = (x0 + (double)i * dx) - ax[p];
            by[p] = (y0 + (double)j * dx) - ay[p];
        }
}

static double min3(double a, double b, double c) { return fmin(fmin(a, b), c); }
static double max3(double a, double b, double c) { return fmax(fmax(a, b), c); }

/* Reading R22: S is inside the closed triangle ABC iff it lies in the closed bounding box of
 * the three vertices AND d != 0, u >= 0, v >= 0, u + v <= 1.  The box is part of the definition: a point of a
 * closed triangle is always inside the box of its vertices, but the ROUNDED barycentric test alone can accept a
 * point one ulp outside an extreme vertex (S - A rounds to B - A, u = 1, v = 0); the box makes that case a miss. */
static int tri_test(const double A[2], const double B[2], const double C[2], const double S[2], double *u, double *v) {
    if (S[0] < min3(A[0], B[0], C[0]) || S[0] > max3(A[0], B[0], C[0]) || S[1] < min3(A[1], B[1], C[1]) ||
        S[1] > max3(A[1], B[1], C[1]))
        return 0;
    const double e1x = B[0] - A[0], e1y = B[1] - A[1];
    const double e2x = C[0] - A[0], e2y = C[1] - A[1];
    const double sx = S[0] - A[0], sy = S[1] - A[1];
    const double d = e1x * e2y - e1y * e2x;
    if (d == 0.0) return 0;
    *u = (sx * e2y - sy * e2x) / d;
    *v = (e1x * sy - e1y * sx) / d;
    return *u >= 0.0 && *v >= 0.0 && *u + *v <= 1.0;
}

/* returns the number of images found (may exceed max_images; only the first max_images are stored) */
long long orc_delens(const double *ax, const double *ay, double x0, double y0, double dx, int nx, int ny,
                     const double *sources /* [ns][2] */, int ns, orc_image *images, long long max_images) {
    long long found = 0;
    for (int j = 0; j + 1 < ny; ++j)
        for (int i = 0; i + 1 < nx; ++i) {
            double T[4][2], Bq[4][2]; /* 00, 10, 01, 11: image-plane and source-plane corners */
            for (int c = 0; c < 4; ++c) {
                const int ii = i + (c & 1), jj = j + (c >> 1);
                const size_t p = (size_t)jj * (size_t)nx + (size_t)ii;
                T[c][0] = x0 + (double)ii * dx;
                T[c][1] = y0 + (double)jj * dx;
                Bq[c][0] = T[c][0] - ax[p];
                Bq[c][1] = T[c][1] - ay[p];
            }
            static const int V[2][3] = {{0, 1, 2}, {3, 2, 1}};
            for (int t = 0; t < 2; ++t)
                for (int s = 0; s < ns; ++s) {
                    double u, v;
                    const int a = V[t][0], b = V[t][1], c = V[t][2];
                    if (!tri_test(Bq[a], Bq[b], Bq[c], &sources[2 * s], &u, &v)) continue;
                    if (found < max_images) {
                        orc_image *im = &images[found];
                        im->source = s;
                        im->pad_ = 0;
                        im->triangle = 2 * ((int64_t)j * (nx - 1) + i) + t;
                        im->x = T[a][0] + u * (T[b][0] - T[a][0]) + v * (T[c][0] - T[a][0]);
                        im->y = T[a][1] + u * (T[b][1] - T[a][1]) + v * (T[c][1] - T[a][1]);
                    }
                    ++found;
                }
        }
    return found;
}

/*
 * ---- NEXT row f3: chi^2 of multiple-image constraints ---------------------------------------
 * "Each image is unlensed onto the source-plane using the mass-model to be tested ... Sending back the
 * barycentre of these positions to the image plane (see Fig. 3), we can define a cost-function
 *   chi^2 = sum_i sum_j (c_ij - x_ij)^2 / sigma_ij^2"                  PAPER.md:76-81 (Fig. 3, eq. 6)
 * Four stages (sec. 4.2): gradient on the grid; sources from the constraints; images
 * by delensing and checking the grid; "the master CPU assigns them to their closest constraint and then
 * computes the chi^2".  Readings R23, the paper being silent on each:
 *   - beta_k = c_k - alpha(c_k) with alpha evaluated AT the constraint (not interpolated on the grid);
 *   - source i = arithmetic mean of the beta_k of its constraints (Fig. 3 "barycentre"); a source
 *     without constraints is ignored;
 *   - predicted images of all sources by orc_delens on the grid;
 *   - x_k = the predicted image of source s_k closest to c_k (so every constraint gets its closest
 *     image; an image may serve several constraints or none);
 *   - a constraint whose source has no predicted image on the grid contributes +infinity;
 *   - (c - x)^2 is the squared Euclidean distance; the sum runs over the constraints in index order.
 */
#include <stdlib.h>

typedef struct {
    int32_t source; /* 0 .. nsources-1 */
    int32_t pad_;
    double x, y;    /* observed image position c_k */
    double sigma;   /* > 0 */
} orc_constraint;

/* returns chi^2; sources_out [nsources][2] and predicted [K][2] may be NULL; *nimages = images found */
double orc_chi2(const orc_lens *lenses, int nlens, double x0, double y0, double dx, int nx, int ny,
                const orc_constraint *c, int K, int nsources, double *sources_out, double *predicted,
                long long *nimages) {
    double *src = (double *)calloc((size_t)(nsources > 0 ? nsources : 1) * 2, sizeof(double));
    int *cnt = (int *)calloc((size_t)(nsources > 0 ? nsources : 1), sizeof(int));
    /* stage 2: unlens the constraints, barycentre per source */
    for (int k = 0; k < K; ++k) {
        orc_deriv d;
        orc_point(lenses, nlens, c[k].x, c[k].y, &d);
        src[2 * c[k].source] += c[k].x - d.ax;
        src[2 * c[k].source + 1] += c[k].y - d.ay;
        cnt[c[k].source] += 1;
    }
    for (int i = 0; i < nsources; ++i) {
        if (cnt[i] > 0) {
            src[2 * i] /= (double)cnt[i];
            src[2 * i + 1] /= (double)cnt[i];
        } else {
            src[2 * i] = src[2 * i + 1] = NAN; /* never inside a triangle */
        }
    }
    /* stage 1: deflection on the grid */
    const size_t np = (size_t)nx * (size_t)ny;
    double *ax = (double *)malloc(np * sizeof(double)), *ay = (double *)malloc(np * sizeof(double));
    orc_planes pl = {ax, ay, NULL, NULL, NULL, NULL, NULL, NULL, NULL};
    orc_grid_rows(lenses, nlens, x0, y0, dx, nx, ny, 0, ny, &pl);
    /* stage 3: predicted images */
    long long cap = 64;
    orc_image *im = (orc_image *)malloc((size_t)cap * sizeof(orc_image));
    long long found = orc_delens(ax, ay, x0, y0, dx, nx, ny, src, nsources, im, cap);
    if (found > cap) {
        cap = found;
        free(im);
        im = (orc_image *)malloc((size_t)cap * sizeof(orc_image));
        found = orc_delens(ax, ay, x0, y0, dx, nx, ny, src, nsources, im, cap);
    }
    /* stage 4: closest image of the same source, chi^2 */
    double chi2 = 0.0;
    for (int k = 0; k < K; ++k) {
        double best = INFINITY, bx = NAN, by = NAN;
        for (long long m = 0; m < found; ++m) {
            if (im[m].source != c[k].source) continue;
            const double ex = c[k].x - im[m].x, ey = c[k].y - im[m].y;
            const double d2 = ex * ex + ey * ey;
            if (d2 < best) { best = d2; bx = im[m].x; by = im[m].y; }
        }
        if (predicted) { predicted[2 * k] = bx; predicted[2 * k + 1] = by; }
        chi2 += best / (c[k].sigma * c[k].sigma);
    }
    if (sources_out)
        for (int i = 0; i < 2 * nsources; ++i) sources_out[i] = src[i];
    if (nimages) *nimages = found;
    free(im); free(ax); free(ay); free(cnt); free(src);
    return chi2;
}

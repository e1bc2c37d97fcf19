// lh_pack.cpp -- host side of step a1: validate the boundary AoS and precompute the
// per-lens constants (O(nlens), double precision, plain C++; no CUDA in here).
#include "lh_pack.h"

#include <cmath>
#include <cstdio>
#include <cstring>

#include "../../include/lh.h"

namespace lh {

static bool finite_all(const lh_lens &L) {
    return std::isfinite(L.x) && std::isfinite(L.y) && std::isfinite(L.ellipticity) && std::isfinite(L.theta) &&
           std::isfinite(L.rcore) && std::isfinite(L.rcut) && std::isfinite(L.b0);
}

static int classify(const lh_lens &L, int idx, int model, char *err, int errlen) {
    auto fail = [&](const char *why) {
        std::snprintf(err, errlen, "lens %d of model %d: %s", idx, model, why);
        return -1;
    };
    if (L.type != LH_DPIE && L.type != LH_NSIE && L.type != LH_SIS) return fail("unknown type");
    if (L.type == LH_SIS) {
        // ellipticity, theta, rcore, rcut are ignored for an SIS (reading 8c-19) -- only what is used must be finite
        if (!(std::isfinite(L.x) && std::isfinite(L.y) && std::isfinite(L.b0))) return fail("non-finite parameter");
        if (!(L.b0 >= 0.0)) return fail("b0 must be >= 0");
        return CLS_SIS;
    }
    if (L.type == LH_NSIE) {
        if (!(std::isfinite(L.x) && std::isfinite(L.y) && std::isfinite(L.ellipticity) && std::isfinite(L.theta) &&
              std::isfinite(L.rcore) && std::isfinite(L.b0)))
            return fail("non-finite parameter");
    } else if (!finite_all(L)) {
        return fail("non-finite parameter");
    }
    if (!(L.b0 >= 0.0)) return fail("b0 must be >= 0");
    if (!(L.ellipticity >= 0.0 && L.ellipticity < 1.0)) return fail("ellipticity outside [0,1)");
    if (!(L.rcore > 0.0)) return fail("rcore must be > 0");
    if (L.type == LH_DPIE && !(L.rcut > L.rcore)) return fail("dPIE needs rcut > rcore");
    const double e = L.ellipticity;
    if (e / (1.0 + std::sqrt(1.0 - e * e)) > EXTREME_EPS) return CLS_EXTREME;
    return L.type == LH_DPIE ? CLS_DPIE : CLS_NSIE;
}

static void fill(const lh_lens &L, int cls, LensK &K) {
    std::memset(&K, 0, sizeof(K));
    K.xc = L.x;
    K.yc = L.y;
    if (cls == CLS_SIS) {
        K.G = K.T = L.b0;
        K.c = 1.0;
        return;
    }
    const double e = L.ellipticity;
    const double eps = e / (1.0 + std::sqrt(1.0 - e * e));  // reading R2
    const double o = 1.0 - eps * eps, p = (1.0 + eps) * (1.0 + eps), m = (1.0 - eps) * (1.0 - eps);
    const double rc = L.rcore;
    const bool cut = (L.type == LH_DPIE);
    const double rt = cut ? L.rcut : 0.0;
    const double T = cut ? L.b0 * rt / (rt - rc) : L.b0;
    // eps -> 0 is taken by never letting 2 sqrt(eps) fall below 2^-40: the scaled frame then makes x'^2
    // vanish against P^_c P^_t exactly (atan(u) = u below 1e-8) and every product stays far inside the
    // double range; the deviation from the true tiny eps is O(2^-82) relative.
    const double sg = std::fmax(2.0 * std::sqrt(eps), 0x1p-40);
    const double k = o / sg;
    const double c2 = std::cos(2.0 * L.theta), s2 = std::sin(2.0 * L.theta);
    K.c = std::cos(L.theta);
    K.s = std::sin(L.theta);
    K.ip = k * k / p;
    K.im = k * k / m;
    K.rc2 = k * k * rc * rc;
    K.rt2 = k * k * rt * rt;
    K.ac = p / sg * rc;
    K.at = p / sg * rt;
    K.bc = m / sg * rc;
    K.bt = m / sg * rt;
    K.G = T * k;
    K.cG = K.c * K.G;
    K.sG = K.s * K.G;
    K.TF = T * k * p / (sg * sg);
    K.r2c = rc * rc;
    K.r2t = rt * rt;
    K.KTF = -4.0 * eps * c2 * K.TF;
    K.K2TF = -2.0 * eps * s2 * K.TF;
    K.dr2 = k * k * (rt * rt - rc * rc);
    K.eps = eps;
    K.sg = sg;
    K.T = T;
}

int pack_model(const void *records, int n, LensK *out, ModelRanges *ranges, char *err, int errlen, int model) {
    const lh_lens *L = static_cast<const lh_lens *>(records);
    int count[CLS_COUNT] = {0, 0, 0, 0};
    // pass 1: validate + count (stable counting sort keeps index order inside a class)
    for (int i = 0; i < n; ++i) {
        int cls = classify(L[i], i, model, err, errlen);
        if (cls < 0) return -1;
        ++count[cls];
    }
    int pos[CLS_COUNT];
    ranges->begin[0] = 0;
    for (int k = 0; k < CLS_COUNT; ++k) {
        pos[k] = ranges->begin[k];
        ranges->begin[k + 1] = ranges->begin[k] + count[k];
    }
    for (int i = 0; i < n; ++i) {
        int cls = classify(L[i], i, model, err, errlen);
        fill(L[i], cls, out[pos[cls]++]);
    }
    return 0;
}

}  // namespace lh

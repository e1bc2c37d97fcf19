// lh_pack.h -- device-side lens table produced by the host packer (a1 in DESIGN.md sec. 1).
//
// The boundary takes an AoS of raw parameters (lh_lens); the device wants, per
// lens, the constants that do not depend on the pixel.  PAPER.md:151 (sec. 3.2.1)
// argues for SoA so that SIMD lanes over *lenses* load homogeneous data; on the
// GPU the lanes run over *pixels* and every lane of a warp needs the same lens at
// the same time, so the right layout is one contiguous record per lens.  The records of
// a launch travel BY VALUE in the kernel parameters (constant bank 0, lh_kernels.h) and
// reach the FP64 instructions as uniform-register operands (LDCU), one field each.
#pragma once
#include <cstdint>

namespace lh {

// Evaluation classes (the table is sorted by class so each inner loop is type-pure).
enum LensClass : int {
    CLS_DPIE = 0,  // dPIE, merged one-atan/one-atanh form
    CLS_NSIE = 1,  // single PIEMD term
    CLS_SIS = 2,   // singular isothermal sphere
    CLS_EXTREME = 3,  // dPIE / NSIE with eps > EXTREME_EPS: two-term form with IEEE sqrt / div and libdevice
                      // atan / atanh, outside the table range of the fast atanh (lh_math.cuh)
    CLS_COUNT = 4
};

// Above this eps = (1-q)/(1+q) the atanh argument u = 2 sqrt(eps)/(1+eps) comes so close to 1 that the fast
// atanh's index argument t = 1 - u, formed with an ABSOLUTE error of u 2^-19.9 (lh_math.cuh), is no longer
// good to a small fraction of its bin: eps = 0.85 <-> e-hat = 0.987 <-> axis ratio q = 0.081 <-> t >= 3.3e-3
// (index error < 3 % of the bin half-width); the table itself would reach to t = 2^-16.
constexpr double EXTREME_EPS = 0.85;

// Notation: eps = e/(1+sqrt(1-e^2)), o = 1-eps^2, p = (1+eps)^2, m = (1-eps)^2,
// sg = 2 sqrt(eps) (never below 2^-40, which takes the circular limit), k = o/sg,
// T = b0*rt/(rt-rc) (dPIE) or b0 (NSIE, SIS), c/s = cos/sin(theta).
// All lengths of the lens frame are carried scaled by k (w^ = k w), which removes the
// 2 sqrt(eps) factors from the atan / atanh arguments (sec. 5.2) and turns D_r into
// (sg^2/p)(P^_r^2 + x'^2) (sec. 5.3); every FP64 instruction of the kernel takes at most ONE field.
struct alignas(16) LensK {
    double xc, yc;      //  0  centre
    double c, s;        //  2  cos(theta), sin(theta)
    double ip, im;      //  4  k^2/p, k^2/m          -> rho^^2 = ip x'^2 + im y'^2
    double rc2, rt2;    //  6  k^2 rcore^2, k^2 rcut^2 -> w^_r = sqrt(r2 + rho^^2); rt2 = 0 marks an NSIE in CLS_EXTREME
    double ac, at;      //  8  (p/sg) rcore, (p/sg) rcut -> P^_r = w^_r + a_r
    double bc, bt;      // 10  (m/sg) rcore, (m/sg) rcut -> Q^_r = w^_r + b_r
    double cG, sG;      // 12  cos, sin(theta) * G
    double G, TF;       // 14  G = T k (also the weight of 1/w^_c - 1/w^_t; SIS: b0);  TF = T k p / sg^2 (weight of f^_r)
    double r2c, r2t;    // 16  rcore^2, rcut^2 (unscaled)
    double KTF, K2TF;   // 18  -4 eps cos(2 theta) TF, -2 eps sin(2 theta) TF
    double dr2, eps;    // 20  k^2 (rcut^2 - rcore^2) = rt2 - rc2;  eps (diagnostic)
    double sg, T;       // 22  diagnostic
};
static_assert(sizeof(LensK) == 24 * 8, "LensK is 24 doubles");
constexpr int LENSK_DOUBLES = sizeof(LensK) / 8;

// Per-model class boundaries inside that model's slice of the table:
// class k occupies [begin[k], begin[k+1]).
struct ModelRanges {
    int32_t begin[CLS_COUNT + 1];
};

// Host: validate `n` boundary records (include/lh.h rules) and fill `out[n]` sorted
// by class, `ranges` for this model.  Returns 0 or writes a message into err.
int pack_model(const void *lh_lens_records, int n, LensK *out, ModelRanges *ranges, char *err, int errlen,
               int model_index);

}  // namespace lh

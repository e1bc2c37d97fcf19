// lh_pack.h -- device-side lens table produced by the host packer (a1 in DESIGN.md sec. 1).
//
// The boundary takes an AoS of raw parameters (lh_lens); the device wants, per
// lens, the constants that do not depend on the pixel.  PAPER.md:151 (sec. 3.2.1)
// argues for SoA so that SIMD lanes over *lenses* load homogeneous data; on the
// GPU the lanes run over *pixels* and every lane of a warp needs the same lens at
// the same time, so the right layout is one contiguous, 16-byte aligned record
// per lens that a warp fetches from shared memory as broadcast 128-bit loads.
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

// Above this eps = (1-q)/(1+q) the ratio (1+u)/(1-u), u = 2 sqrt(eps)/(1+eps), approaches the 2^16 end
// of the atanh table: eps = 0.96 <-> e-hat = 0.99917 <-> axis ratio q = 0.0204 <-> ratio < 9700.
constexpr double EXTREME_EPS = 0.96;

// Notation: eps = e/(1+sqrt(1-e^2)), o = 1-eps^2, p = (1+eps)^2,
// m = (1-eps)^2, T = b0*rt/(rt-rc) (dPIE) or b0 (NSIE, SIS), c/s = cos/sin(theta).
// The gradient constants are those of sec. 5.2 divided by o, so that every FP64 instruction of
// the kernel takes at most ONE of these (uniform-register) fields.
struct alignas(16) LensK {
    double xc, yc;      //  0  centre
    double c, s;        //  2  cos(theta), sin(theta)
    double ip, im;      //  4  1/p, 1/m              -> rho^2 = ip x'^2 + im y'^2
    double rc2, rt2;    //  6  rcore^2, rcut^2       -> w_r = sqrt(r^2 + rho^2); rt2 = 0 marks an NSIE in CLS_EXTREME
    double o, se;       //  8  1-eps^2; 2 sqrt(eps)/o, replaced by 2^-500 when eps == 0
    double ac, at;      // 10  (p/o) rcore, (p/o) rcut   -> P_r = w_r + a_r
    double bc, bt;      // 12  (m/o) rcore, (m/o) rcut   -> Q_r = w_r + b_r
    double cG, sG;      // 14  cos, sin(theta) * G,  G = T / se
    double T, eps;      // 16  T; eps (diagnostic)
    double orc2, ort2;  // 18  2 o rcore, 2 o rcut   -> D_r = c0_r + R^2 + (2 o r) w_r
    double c0c, c0t;    // 20  2 (1+eps^2) r^2
    double KT, K2T;     // 22  -4 eps cos(2 theta) T, -2 eps sin(2 theta) T
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

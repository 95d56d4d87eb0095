// nn_relax.cuh -- per-neuron linear relaxations  kL z + bL <= phi(z) <= kU z + bU  on [l, u]
// (the activation step of CROWN, Thm 2 / eq. (18); the paper cites [26] and
// gives no formulas -- DESIGN.md readings R8/R9), in "deviation form":
//     gU = kU zhat + bU - phi(zhat) >= 0,   gL = kL zhat + bL - phi(zhat) <= 0
// are the gaps of the two lines at the nominal pre-activation zhat.  O(width) work per layer, so it
// is done in FP64 (removes the per-neuron cancellations) and stored as FP32.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace leb_nn {

constexpr int ACT_RELU = 1, ACT_TANH = 2;
constexpr int kBisect = 52;
constexpr double kTanhD2Max = 0.76980035891950104;   // max |tanh''| = 4 / (3 sqrt 3)
constexpr double kDegenerate = 1e-12;

// how each line was built (needed again by the VJP)
enum { LINE_ZERO = 0, LINE_IDENT, LINE_CHORD, LINE_TAN_MID, LINE_TAN_IMPL, LINE_RELU_LOW, LINE_DEGEN };

struct Relax {
    double kU, bU, kL, bL;
    int cU, cL;        // LINE_* of the upper / lower line
    double dU, dL;     // tangent points where applicable
    double tl, tu;     // tanh(l), tanh(u) (tanh only; the VJP reuses them instead of evaluating tanh again)
};

__device__ __forceinline__ double th(double x) { return tanh(x); }
__device__ __forceinline__ double th1(double x) { double t = tanh(x); return 1.0 - t * t; }
__device__ __forceinline__ double th2(double x) { double t = tanh(x); return -2.0 * t * (1.0 - t * t); }

__device__ inline Relax relax_relu(double l, double u) {
    Relax r{};
    if (u <= 0.0) { r.cU = r.cL = LINE_ZERO; return r; }
    if (l >= 0.0) { r.kU = r.kL = 1.0; r.cU = r.cL = LINE_IDENT; return r; }
    double w = u - l;
    r.kU = u / w;
    r.bU = -u * l / w;
    r.cU = LINE_CHORD;
    r.kL = (u > -l) ? 1.0 : 0.0;     // adaptive lower slope; tie u == -l -> 0 (reading R8)
    r.bL = 0.0;
    r.cL = LINE_RELU_LOW;
    return r;
}

// tangent point of the upper line through (l, tanh l), l < 0 < u: root of
// h(d) = t'(d)(d - l) - (t(d) - t(l)) on (0, u); h > 0 left of the root.  Returns the bracket end
// d >= d*, the side on which the tangent stays above tanh on [l, u] (sound side).
// The bracket [a, b] keeps h(a) > 0 >= h(b) as in a bisection -- whatever is returned was evaluated with h <= 0 -- but the
// points are chosen better: the first is -l / 2 (the exact tangent point for the cubic z - z^3 / 3, which tanh is near 0:
// without it the iteration from u only converges linearly while |l| << d), then Newton steps from b
// (h'(d) = t''(d)(d - l)), shortened by 2^-20 so that near the root they stay on that side; a step that leaves the bracket
// is replaced by the secant point, then by the midpoint.  Ends when b no longer moves by 2^-48 of itself: 7 evaluations of
// tanh on average and 12 at the 99th percentile instead of 52 -- every lane of a warp waits for the slowest, and at
// config 5 nearly every warp holds a mixed-sign neuron.  kBisect bounds the loop.
__device__ __forceinline__ void tangent_h(double m, double l, double tl, double& h, double& dh) {
    const double t = tanh(m), s = 1.0 - t * t;
    h = s * (m - l) - (t - tl);
    dh = -2.0 * t * s * (m - l);
}
__device__ inline double tangent_upper(double l, double u, double tl) {
    constexpr double kShort = 0.99999904632568359375, kTol = 3.5527136788005009e-15;      // 1 - 2^-20, 2^-48
    double a = 0.0, ha = tl - l;                 // h(0) = tanh(l) - l > 0
    double b = u, hb, db;
    tangent_h(b, l, tl, hb, db);
    const double g = -0.5 * l;
    if (g < b) {
        double hg, dg;
        tangent_h(g, l, tl, hg, dg);
        if (hg > 0.0) { a = g; ha = hg; } else { b = g; hb = hg; db = dg; }
    }
    for (int it = 0; it < kBisect; ++it) {
        if (!(b - a > kTol * b)) break;
        const double step = (hb / db) * kShort;
        if (!(step > kTol * b)) break;
        double m = b - step;
        if (!(m > a)) {
            m = a + (b - a) * (ha / (ha - hb));
            if (!(m > a && m < b)) {
                m = 0.5 * (a + b);
                if (!(m > a && m < b)) break;
            }
        }
        double hm, dm;
        tangent_h(m, l, tl, hm, dm);
        if (hm > 0.0) { a = m; ha = hm; } else { b = m; hb = hm; db = dm; }
    }
    return b;
}
// tangent point of the lower line through (u, tanh u), in (l, 0): the mirror image (tanh is odd).  Returns the end
// d <= d* (sound side).
__device__ inline double tangent_lower(double l, double u, double tu) { return -tangent_upper(-u, -l, -tu); }

__device__ inline Relax relax_tanh(double l, double u) {
    Relax r{};
    double w = u - l;
    if (w < kDegenerate) {           // point interval: tangent at the midpoint, widened by the curvature bound
        double d = 0.5 * (l + u), k = th1(d), b = th(d) - k * d, e = 0.5 * kTanhD2Max * w * w;
        r.kU = r.kL = k; r.bU = b + e; r.bL = b - e; r.cU = r.cL = LINE_DEGEN; r.dU = r.dL = d;
        return r;
    }
    double tl = th(l), tu = th(u);
    r.tl = tl; r.tu = tu;
    double kc = (tu - tl) / w, bc = tl - kc * l;
    if (l >= 0.0) {                  // concave part: tangent above, chord below
        double d = 0.5 * (l + u), k = th1(d);
        r.kU = k; r.bU = th(d) - k * d; r.cU = LINE_TAN_MID; r.dU = d;
        r.kL = kc; r.bL = bc; r.cL = LINE_CHORD;
        return r;
    }
    if (u <= 0.0) {                  // convex part: chord above, tangent below
        double d = 0.5 * (l + u), k = th1(d);
        r.kL = k; r.bL = th(d) - k * d; r.cL = LINE_TAN_MID; r.dL = d;
        r.kU = kc; r.bU = bc; r.cU = LINE_CHORD;
        return r;
    }
    if (kc <= 1.0 - tu * tu) { r.kU = kc; r.bU = bc; r.cU = LINE_CHORD; }
    else { double d = tangent_upper(l, u, tl), k = th1(d); r.kU = k; r.bU = th(d) - k * d; r.cU = LINE_TAN_IMPL; r.dU = d; }
    if (kc <= 1.0 - tl * tl) { r.kL = kc; r.bL = bc; r.cL = LINE_CHORD; }
    else { double d = tangent_lower(l, u, tu), k = th1(d); r.kL = k; r.bL = th(d) - k * d; r.cL = LINE_TAN_IMPL; r.dL = d; }
    return r;
}

__device__ inline Relax relax_any(int act, double l, double u) { return act == ACT_RELU ? relax_relu(l, u) : relax_tanh(l, u); }

__device__ __forceinline__ double act_f(int act, double z) { return act == ACT_RELU ? fmax(z, 0.0) : tanh(z); }
__device__ __forceinline__ double act_d1(int act, double z) { return act == ACT_RELU ? (z > 0.0 ? 1.0 : 0.0) : th1(z); }   // phi'(0)=0 (R12)
__device__ __forceinline__ double act_d2(int act, double z) { return act == ACT_RELU ? 0.0 : th2(z); }

// Adjoint of one line's (k, b) with respect to (l, u):  (lb, ub) += d(k,b)/d(l,u)^T (kb, bb).
// tl, tu = tanh(l), tanh(u) as relax_tanh computed them (Relax::tl, tu).
__device__ inline void line_vjp(int act, int how, bool upper, double l, double u, double d, double kb, double bb,
                                double& lb, double& ub, double tl, double tu) {
    switch (how) {
        case LINE_CHORD: {
            double w = u - l;
            if (act == ACT_RELU) {      // k = u/(u-l), b = -u l/(u-l)
                double w2 = w * w;
                lb += kb * (u / w2) + bb * (-u * u / w2);
                ub += kb * (-l / w2) + bb * (l * l / w2);
            } else {                    // k = (t(u)-t(l))/(u-l), b = t(l) - k l
                double k = (tu - tl) / w;
                double t1l = 1.0 - tl * tl, t1u = 1.0 - tu * tu;
                double dk_du = (t1u - k) / w, dk_dl = (k - t1l) / w;
                double db_dl = t1l - k - l * dk_dl, db_du = -l * dk_du;
                lb += kb * dk_dl + bb * db_dl;
                ub += kb * dk_du + bb * db_du;
            }
            break;
        }
        case LINE_TAN_MID: {            // k = t'(d), b = t(d) - t'(d) d, d = (l+u)/2
            double ad = th2(d) * (kb - d * bb);
            lb += 0.5 * ad;
            ub += 0.5 * ad;
            break;
        }
        case LINE_TAN_IMPL: {           // tangent point defined implicitly by l (upper) or by u (lower)
            const double td = tanh(d), t1d = 1.0 - td * td, t2d = -2.0 * td * t1d;
            double ad = t2d * (kb - d * bb);
            if (upper) lb += ad * (t1d - (1.0 - tl * tl)) / (t2d * (d - l));
            else ub += ad * ((1.0 - tu * tu) - t1d) / (t2d * (u - d));
            break;
        }
        case LINE_DEGEN: {              // b = t(d) - k d +- c (u-l)^2, c = kTanhD2Max/2
            double ad = th2(d) * (kb - d * bb);
            double dw = kTanhD2Max * (u - l) * bb * (upper ? 1.0 : -1.0);
            lb += 0.5 * ad - dw;
            ub += 0.5 * ad + dw;
            break;
        }
        default: break;                 // LINE_ZERO, LINE_IDENT, LINE_RELU_LOW: constants
    }
}

}  // namespace leb_nn

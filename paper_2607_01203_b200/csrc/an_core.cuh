// an_core.cuh -- FP32 outward-rounded interval arithmetic, second-order interval jets and the
// analytic model straight-line programs (SLPs) for the path-based interval-Hessian bound
// (Thm 1, eq. (15)).  Device code of the product; shares nothing with oracle/.
//
// Inclusion-function contract (reading R1): [H_{l,kj}](box) is the natural interval
// extension of second-order forward-mode AD of the model SLP in directions (e_j, e_k); every SLP
// variable carries intervals (w, w_j, w_k, w_jk).  Interval * is the hull of the four endpoint
// products, sqr is non-negative, sin/cos are range-exact.  All lower endpoints are rounded
// towards -inf and all upper endpoints towards +inf (FADD/FMUL/FFMA .RM/.RP run at full rate),
// sinf/cosf are padded outward by their documented 2-ulp error bound, so every enclosure
// computed here contains the exact-arithmetic one.
//
// Scalar type S is `float` (forward) or `Du` (value + one tangent, VJP by forward-mode duals:
// min/max/abs select a branch by value, ties take the first candidate in the order
// lo*lo, lo*hi, hi*lo, hi*hi -- DESIGN.md "VJP definition").
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#if defined(__CUDA_ARCH__)
#define LEB_HD __host__ __device__ __forceinline__
#else
#define LEB_HD inline
#endif

namespace leb_an {

// ------------------------------------------------------------------ directed rounding (float)
#if defined(__CUDA_ARCH__)
LEB_HD float add_dn(float a, float b) { return __fadd_rd(a, b); }
LEB_HD float add_up(float a, float b) { return __fadd_ru(a, b); }
LEB_HD float mul_dn(float a, float b) { return __fmul_rd(a, b); }
LEB_HD float mul_up(float a, float b) { return __fmul_ru(a, b); }
LEB_HD float rcp_dn(float a) { return __frcp_rd(a); }
LEB_HD float rcp_up(float a) { return __frcp_ru(a); }
#else
// Host build (debug emulation under _work/ only; the product never runs this): round the exact
// double result outward to float.
inline float dn_(double x) { float f = (float)x; return ((double)f > x) ? nextafterf(f, -INFINITY) : f; }
inline float up_(double x) { float f = (float)x; return ((double)f < x) ? nextafterf(f, INFINITY) : f; }
inline float add_dn(float a, float b) { return dn_((double)a + (double)b); }
inline float add_up(float a, float b) { return up_((double)a + (double)b); }
inline float mul_dn(float a, float b) { return dn_((double)a * (double)b); }
inline float mul_up(float a, float b) { return up_((double)a * (double)b); }
inline float rcp_dn(float a) { return dn_(1.0 / (double)a); }
inline float rcp_up(float a) { return up_(1.0 / (double)a); }
#endif

// ------------------------------------------------------------------ dual scalar
struct Du { float v, d; };

LEB_HD float val(float x) { return x; }
LEB_HD float val(const Du& x) { return x.v; }
LEB_HD float tan_(float) { return 0.f; }
LEB_HD float tan_(const Du& x) { return x.d; }
template <class S> LEB_HD S mk(float v);
template <> LEB_HD float mk<float>(float v) { return v; }
template <> LEB_HD Du mk<Du>(float v) { return Du{v, 0.f}; }

LEB_HD Du add_dn(Du a, Du b) { return {add_dn(a.v, b.v), a.d + b.d}; }
LEB_HD Du add_up(Du a, Du b) { return {add_up(a.v, b.v), a.d + b.d}; }
LEB_HD Du mul_dn(Du a, Du b) { return {mul_dn(a.v, b.v), fmaf(a.d, b.v, a.v * b.d)}; }
LEB_HD Du mul_up(Du a, Du b) { return {mul_up(a.v, b.v), fmaf(a.d, b.v, a.v * b.d)}; }
LEB_HD float neg(float a) { return -a; }
LEB_HD Du neg(Du a) { return {-a.v, -a.d}; }
// scale by a plain constant c
LEB_HD float cmul_dn(float c, float a) { return mul_dn(c, a); }
LEB_HD float cmul_up(float c, float a) { return mul_up(c, a); }
LEB_HD Du cmul_dn(float c, Du a) { return {mul_dn(c, a.v), c * a.d}; }
LEB_HD Du cmul_up(float c, Du a) { return {mul_up(c, a.v), c * a.d}; }
// 1/a : d(1/a) = -a'/a^2
LEB_HD Du rcp_dn(Du a) { float r = rcp_dn(a.v); return {r, -a.d * r * r}; }
LEB_HD Du rcp_up(Du a) { float r = rcp_up(a.v); return {r, -a.d * r * r}; }
// branch selection by value; ties keep the first argument
template <class S> LEB_HD S min1(S a, S b) { return val(b) < val(a) ? b : a; }
template <class S> LEB_HD S max1(S a, S b) { return val(b) > val(a) ? b : a; }

// sin / cos endpoint values with an outward pad covering the 2-ulp error of sinf / cosf
LEB_HD float pad_dn(float s) { return fmaxf(-1.f, add_dn(s, -(fabsf(s) * 3.0e-7f + 1e-30f))); }
LEB_HD float pad_up(float s) { return fminf(1.f, add_up(s, (fabsf(s) * 3.0e-7f + 1e-30f))); }
LEB_HD float sin_dn(float x) { return pad_dn(sinf(x)); }
LEB_HD float sin_up(float x) { return pad_up(sinf(x)); }
LEB_HD float cos_dn(float x) { return pad_dn(cosf(x)); }
LEB_HD float cos_up(float x) { return pad_up(cosf(x)); }
LEB_HD Du sin_dn(Du x) { return {sin_dn(x.v), cosf(x.v) * x.d}; }
LEB_HD Du sin_up(Du x) { return {sin_up(x.v), cosf(x.v) * x.d}; }
LEB_HD Du cos_dn(Du x) { return {cos_dn(x.v), -sinf(x.v) * x.d}; }
LEB_HD Du cos_up(Du x) { return {cos_up(x.v), -sinf(x.v) * x.d}; }

// ------------------------------------------------------------------ intervals
template <class S> struct Iv { S lo, hi; };

template <class S> LEB_HD Iv<S> iconst(float c) { return {mk<S>(c), mk<S>(c)}; }
template <class S> LEB_HD Iv<S> iadd(const Iv<S>& a, const Iv<S>& b) { return {add_dn(a.lo, b.lo), add_up(a.hi, b.hi)}; }
template <class S> LEB_HD Iv<S> isub(const Iv<S>& a, const Iv<S>& b) { return {add_dn(a.lo, neg(b.hi)), add_up(a.hi, neg(b.lo))}; }
template <class S> LEB_HD Iv<S> ineg(const Iv<S>& a) { return {neg(a.hi), neg(a.lo)}; }
template <class S> LEB_HD Iv<S> iscale(float c, const Iv<S>& a) {
    if (c >= 0.f) return {cmul_dn(c, a.lo), cmul_up(c, a.hi)};
    return {cmul_dn(c, a.hi), cmul_up(c, a.lo)};
}
template <class S> LEB_HD Iv<S> imul(const Iv<S>& a, const Iv<S>& b) {
    Iv<S> r;
    r.lo = min1(min1(min1(mul_dn(a.lo, b.lo), mul_dn(a.lo, b.hi)), mul_dn(a.hi, b.lo)), mul_dn(a.hi, b.hi));
    r.hi = max1(max1(max1(mul_up(a.lo, b.lo), mul_up(a.lo, b.hi)), mul_up(a.hi, b.lo)), mul_up(a.hi, b.hi));
    return r;
}
template <class S> LEB_HD Iv<S> isqr(const Iv<S>& a) {
    if (val(a.lo) >= 0.f) return {mul_dn(a.lo, a.lo), mul_up(a.hi, a.hi)};
    if (val(a.hi) <= 0.f) return {mul_dn(a.hi, a.hi), mul_up(a.lo, a.lo)};
    return {mk<S>(0.f), max1(mul_up(a.lo, a.lo), mul_up(a.hi, a.hi))};
}
// x^3 is increasing; for x < 0 the lower bound is -(up(|x|^3))
template <class S> LEB_HD S cube_dn(S x) {
    if (val(x) >= 0.f) return mul_dn(mul_dn(x, x), x);
    S m = neg(x);
    return neg(mul_up(mul_up(m, m), m));
}
template <class S> LEB_HD S cube_up(S x) {
    if (val(x) >= 0.f) return mul_up(mul_up(x, x), x);
    S m = neg(x);
    return neg(mul_dn(mul_dn(m, m), m));
}
template <class S> LEB_HD Iv<S> icube(const Iv<S>& a) { return {cube_dn(a.lo), cube_up(a.hi)}; }

// does [lo, hi] contain a point c + 2 pi k ?  (FP64 test with a tiny outward slack: when in doubt
// say yes, which only widens the enclosure by O(slack^2))
LEB_HD bool contains_2pik(float lo, float hi, double c) {
    const double TWO_PI = 6.283185307179586476925286766559;
    double a = ((double)lo - c) / TWO_PI - 1e-9, b = ((double)hi - c) / TWO_PI + 1e-9;
    return floor(b) >= ceil(a);
}
template <class S> LEB_HD Iv<S> isin(const Iv<S>& a) {
    const double HALF_PI = 1.5707963267948966192313216916398;
    bool has_max = contains_2pik(val(a.lo), val(a.hi), HALF_PI);
    bool has_min = contains_2pik(val(a.lo), val(a.hi), -HALF_PI);
    Iv<S> r;
    r.hi = has_max ? mk<S>(1.f) : max1(sin_up(a.lo), sin_up(a.hi));
    r.lo = has_min ? mk<S>(-1.f) : min1(sin_dn(a.lo), sin_dn(a.hi));
    return r;
}
template <class S> LEB_HD Iv<S> icos(const Iv<S>& a) {
    const double PI = 3.1415926535897932384626433832795;
    bool has_max = contains_2pik(val(a.lo), val(a.hi), 0.0);
    bool has_min = contains_2pik(val(a.lo), val(a.hi), PI);
    Iv<S> r;
    r.hi = has_max ? mk<S>(1.f) : max1(cos_up(a.lo), cos_up(a.hi));
    r.lo = has_min ? mk<S>(-1.f) : min1(cos_dn(a.lo), cos_dn(a.hi));
    return r;
}
// 1/a; *bad is raised when 0 is in a (domain error: the enclosure would be unbounded)
template <class S> LEB_HD Iv<S> irecip(const Iv<S>& a, bool* bad) {
    if (val(a.lo) <= 0.f && val(a.hi) >= 0.f) { *bad = true; return iconst<S>(1.f); }
    return {rcp_dn(a.hi), rcp_up(a.lo)};
}

// ------------------------------------------------------------------ second-order jets
template <class S> struct Jet { Iv<S> w, wj, wk, wjk; };

template <class S> LEB_HD Jet<S> jzero() { Iv<S> z = iconst<S>(0.f); return {z, z, z, z}; }
template <class S> LEB_HD Jet<S> jadd(const Jet<S>& a, const Jet<S>& b) {
    return {iadd(a.w, b.w), iadd(a.wj, b.wj), iadd(a.wk, b.wk), iadd(a.wjk, b.wjk)};
}
template <class S> LEB_HD Jet<S> jsub(const Jet<S>& a, const Jet<S>& b) {
    return {isub(a.w, b.w), isub(a.wj, b.wj), isub(a.wk, b.wk), isub(a.wjk, b.wjk)};
}
template <class S> LEB_HD Jet<S> jneg(const Jet<S>& a) { return {ineg(a.w), ineg(a.wj), ineg(a.wk), ineg(a.wjk)}; }
template <class S> LEB_HD Jet<S> jscale(float c, const Jet<S>& a) {
    return {iscale(c, a.w), iscale(c, a.wj), iscale(c, a.wk), iscale(c, a.wjk)};
}
template <class S> LEB_HD Jet<S> jaddc(const Jet<S>& a, float c) {
    Jet<S> r = a;
    r.w = iadd(a.w, iconst<S>(c));
    return r;
}
// product rule; on the diagonal (j == k) the cross term is 2 a_j b_j
template <class S> LEB_HD Jet<S> jmul(const Jet<S>& a, const Jet<S>& b, bool diag) {
    Jet<S> r;
    r.w = imul(a.w, b.w);
    r.wj = iadd(imul(a.wj, b.w), imul(a.w, b.wj));
    r.wk = iadd(imul(a.wk, b.w), imul(a.w, b.wk));
    Iv<S> cross = diag ? iscale(2.f, imul(a.wj, b.wj)) : iadd(imul(a.wj, b.wk), imul(a.wk, b.wj));
    r.wjk = iadd(iadd(imul(a.wjk, b.w), cross), imul(a.w, b.wjk));
    return r;
}
// w = phi(a) from enclosures f, f1, f2 of phi, phi', phi'' on a.w; on the diagonal a_j a_k = sqr(a_j)
template <class S> LEB_HD Jet<S> junary(const Jet<S>& a, const Iv<S>& f, const Iv<S>& f1, const Iv<S>& f2, bool diag) {
    Jet<S> r;
    r.w = f;
    r.wj = imul(f1, a.wj);
    r.wk = imul(f1, a.wk);
    Iv<S> jk = diag ? isqr(a.wj) : imul(a.wj, a.wk);
    r.wjk = iadd(imul(f2, jk), imul(f1, a.wjk));
    return r;
}
template <class S> LEB_HD void jsincos(const Jet<S>& a, bool diag, Jet<S>* s_out, Jet<S>* c_out) {
    Iv<S> s = isin(a.w), c = icos(a.w);
    *s_out = junary(a, s, c, ineg(s), diag);          // (sin)' = cos, (sin)'' = -sin
    *c_out = junary(a, c, ineg(s), ineg(c), diag);    // (cos)' = -sin, (cos)'' = -cos
}
template <class S> LEB_HD Jet<S> jrecip(const Jet<S>& a, bool diag, bool* bad) {
    Iv<S> r = irecip(a.w, bad);
    return junary(a, r, ineg(isqr(r)), iscale(2.f, icube(r)), diag);   // (1/a)' = -1/a^2, (1/a)'' = 2/a^3
}
template <class S> LEB_HD Jet<S> jcube(const Jet<S>& a, bool diag) {
    return junary(a, icube(a.w), iscale(3.f, isqr(a.w)), iscale(6.f, a.w), diag);
}

// ------------------------------------------------------------------ models
struct Model {
    int id, integ, n_units, n, N;
    float dt, half_dt, dt6;                 // dt, dt/2, dt/6
    float inv_m, g, cp, cq, cr, iJx, iJy, iJz;   // 1/m, g, (Jy-Jz)/Jx, (Jz-Jx)/Jy, (Jx-Jy)/Jz, 1/J*
    float k1, k3;
};

// quad12 vector field: xi = (px,py,pz, phi,theta,psi, vx,vy,vz, p,q,r),
// nu = (T, tau_phi, tau_theta, tau_psi); coup (may be NULL) = summed spring force per axis.
template <class S>
LEB_HD void quad12_field(const Model& M, const Jet<S>* xi, const Jet<S>* nu, const Jet<S>* coup, Jet<S>* out,
                         bool diag, bool* bad) {
    Jet<S> sphi, cphi, sth, cth, spsi, cpsi;
    jsincos(xi[3], diag, &sphi, &cphi);
    jsincos(xi[4], diag, &sth, &cth);
    jsincos(xi[5], diag, &spsi, &cpsi);
    Jet<S> rcth = jrecip(cth, diag, bad);
    const Jet<S>&p = xi[9], &q = xi[10], &r = xi[11];
    Jet<S> a = jadd(jmul(q, sphi, diag), jmul(r, cphi, diag));
    out[0] = xi[6];
    out[1] = xi[7];
    out[2] = xi[8];
    out[3] = jadd(p, jmul(a, jmul(sth, rcth, diag), diag));
    out[4] = jsub(jmul(q, cphi, diag), jmul(r, sphi, diag));
    out[5] = jmul(a, rcth, diag);
    Jet<S> Tm = jscale(M.inv_m, nu[0]);
    out[6] = jmul(Tm, jadd(jmul(jmul(cpsi, sth, diag), cphi, diag), jmul(spsi, sphi, diag)), diag);
    out[7] = jmul(Tm, jsub(jmul(jmul(spsi, sth, diag), cphi, diag), jmul(cpsi, sphi, diag)), diag);
    out[8] = jaddc(jmul(Tm, jmul(cth, cphi, diag), diag), -M.g);
    out[9] = jadd(jscale(M.cp, jmul(q, r, diag)), jscale(M.iJx, nu[1]));
    out[10] = jadd(jscale(M.cq, jmul(p, r, diag)), jscale(M.iJy, nu[2]));
    out[11] = jadd(jscale(M.cr, jmul(p, q, diag)), jscale(M.iJz, nu[3]));
    if (coup) {
#pragma unroll
        for (int c = 0; c < 3; ++c) out[6 + c] = jadd(out[6 + c], jscale(M.inv_m, coup[c]));
    }
}

// spring force between unit q (pos pa) and unit q+1 (pos pb), per axis: s = k1 d + k3 d^3, d = pb - pa
template <class S>
LEB_HD Jet<S> spring(const Model& M, const Jet<S>& pa, const Jet<S>& pb, bool diag) {
    Jet<S> d = jsub(pb, pa);
    return jadd(jscale(M.k1, d), jscale(M.k3, jcube(d, diag)));
}

// Input jets of the prefix box A^(j) (eq. (14)): coordinates <= j are the interval
// [nom - rad, nom + rad], coordinates > j are pinned to the nominal point; direction seeds e_j, e_k.
template <class S> struct Inputs {
    const S* nom;   // N scalars (shared memory or registers)
    const S* rad;
    int j, k;
    LEB_HD Jet<S> operator()(int g) const {
        Jet<S> r;
        if (g <= j) r.w = {add_dn(nom[g], neg(rad[g])), add_up(nom[g], rad[g])};
        else r.w = {nom[g], nom[g]};
        r.wj = iconst<S>(g == j ? 1.f : 0.f);
        r.wk = iconst<S>(g == k ? 1.f : 0.f);
        r.wjk = iconst<S>(0.f);
        return r;
    }
};

// f of the centre unit `i` of a quad chain (U = 1: the single quadrotor), all 12 outputs.
// Only the dependency cone of unit i is evaluated: under RK4 the
// stage-1 and stage-2 fields of units i-1, i, i+1, the stage-3/4 fields of unit i, and the
// positions of units i-2 .. i+2 as far as those fields read them.  Every SLP variable that is
// evaluated is evaluated exactly as in the whole-chain SLP, so the enclosures are the same.
template <class S>
LEB_HD void chain_center_f(const Model& M, const Inputs<S>& in, int i, Jet<S>* f, bool* bad) {
    const int U = M.n_units, n = M.n;
    const bool diag = (in.j == in.k);
    const bool hasL = i > 0, hasR = i + 1 < U, hasLL = i > 1, hasRR = i + 2 < U;
    // window slots: 0..4 <-> units i-2 .. i+2 ; full states kept for slots 1..3
    Jet<S> X[3][12], K[3][12], nu[3][4], P[5][3], acc[12], V2[2][3];
    bool ex[5] = {hasLL, hasL, true, hasR, hasRR};
    for (int s = 0; s < 3; ++s) {
        if (!ex[s + 1]) continue;
        int q = i - 1 + s;
        for (int c = 0; c < 12; ++c) X[s][c] = in(12 * q + c);
        for (int c = 0; c < 4; ++c) nu[s][c] = in(n + 4 * q + c);
    }
    for (int s = 0; s < 5; ++s) {
        if (!ex[s]) continue;
        int q = i - 2 + s;
        for (int c = 0; c < 3; ++c) P[s][c] = in(12 * q + c);
    }
    // field of window slot s (1..3) at the current stage, using positions P[] for the springs
    auto field = [&](int s) {
        int q = i - 2 + s;
        bool l = q > 0, r = q + 1 < U;
        Jet<S> coup[3];
        if (l || r) {
            for (int c = 0; c < 3; ++c) {
                if (l && r) coup[c] = jsub(spring(M, P[s][c], P[s + 1][c], diag), spring(M, P[s - 1][c], P[s][c], diag));
                else if (r) coup[c] = spring(M, P[s][c], P[s + 1][c], diag);
                else coup[c] = jneg(spring(M, P[s - 1][c], P[s][c], diag));
            }
        }
        quad12_field(M, X[s - 1], nu[s - 1], (l || r) ? coup : (const Jet<S>*)nullptr, K[s - 1], diag, bad);
    };
    // ---- stage 1
    field(2);
    if (M.integ == 1) {   // forward Euler
        for (int c = 0; c < 12; ++c) f[c] = jadd(in(12 * i + c), jscale(M.dt, K[1][c]));
        return;
    }
    if (hasL) field(1);
    if (hasR) field(3);
    for (int c = 0; c < 12; ++c) acc[c] = K[1][c];
    // ---- stage 2 states: x + (dt/2) k1
    if (hasLL) for (int c = 0; c < 3; ++c) P[0][c] = jadd(P[0][c], jscale(M.half_dt, in(12 * (i - 2) + 6 + c)));
    if (hasRR) for (int c = 0; c < 3; ++c) P[4][c] = jadd(P[4][c], jscale(M.half_dt, in(12 * (i + 2) + 6 + c)));
    for (int s = 0; s < 3; ++s) {
        if (!ex[s + 1]) continue;
        int q = i - 1 + s;
        for (int c = 0; c < 12; ++c) X[s][c] = jadd(in(12 * q + c), jscale(M.half_dt, K[s][c]));
        for (int c = 0; c < 3; ++c) P[s + 1][c] = X[s][c];
    }
    // neighbours' stage-2 velocities = k2[pos] of the neighbours (needed for their stage-3 positions)
    if (hasL) for (int c = 0; c < 3; ++c) V2[0][c] = X[0][6 + c];
    if (hasR) for (int c = 0; c < 3; ++c) V2[1][c] = X[2][6 + c];
    field(2);
    if (hasL) field(1);
    if (hasR) field(3);
    for (int c = 0; c < 12; ++c) acc[c] = jadd(acc[c], jscale(2.f, K[1][c]));
    // ---- stage 3: centre full state x + (dt/2) k2; neighbours: position x + (dt/2) k2[pos] and
    //      velocity x[vel] + (dt/2) k2[vel] (= k3[pos] of the neighbour)
    Jet<S> V3[2][3];
    if (hasL) for (int c = 0; c < 3; ++c) {
        P[1][c] = jadd(in(12 * (i - 1) + c), jscale(M.half_dt, V2[0][c]));
        V3[0][c] = jadd(in(12 * (i - 1) + 6 + c), jscale(M.half_dt, K[0][6 + c]));
    }
    if (hasR) for (int c = 0; c < 3; ++c) {
        P[3][c] = jadd(in(12 * (i + 1) + c), jscale(M.half_dt, V2[1][c]));
        V3[1][c] = jadd(in(12 * (i + 1) + 6 + c), jscale(M.half_dt, K[2][6 + c]));
    }
    for (int c = 0; c < 12; ++c) X[1][c] = jadd(in(12 * i + c), jscale(M.half_dt, K[1][c]));
    for (int c = 0; c < 3; ++c) P[2][c] = X[1][c];
    field(2);
    for (int c = 0; c < 12; ++c) acc[c] = jadd(acc[c], jscale(2.f, K[1][c]));
    // ---- stage 4: x + dt k3
    if (hasL) for (int c = 0; c < 3; ++c) P[1][c] = jadd(in(12 * (i - 1) + c), jscale(M.dt, V3[0][c]));
    if (hasR) for (int c = 0; c < 3; ++c) P[3][c] = jadd(in(12 * (i + 1) + c), jscale(M.dt, V3[1][c]));
    for (int c = 0; c < 12; ++c) X[1][c] = jadd(in(12 * i + c), jscale(M.dt, K[1][c]));
    for (int c = 0; c < 3; ++c) P[2][c] = X[1][c];
    field(2);
    for (int c = 0; c < 12; ++c) {
        acc[c] = jadd(acc[c], K[1][c]);
        f[c] = jadd(in(12 * i + c), jscale(M.dt6, acc[c]));
    }
}

// unicycle (config 1): a = (px, py, th, v, om)
template <class S>
LEB_HD void unicycle_f(const Model& M, const Inputs<S>& in, Jet<S>* f) {
    const bool diag = (in.j == in.k);
    Jet<S> s, c;
    jsincos(in(2), diag, &s, &c);
    f[0] = jadd(in(0), jscale(M.dt, jmul(in(3), c, diag)));
    f[1] = jadd(in(1), jscale(M.dt, jmul(in(3), s, diag)));
    f[2] = jadd(in(2), jscale(M.dt, in(4)));
}

// ------------------------------------------------------------------ window variable lists
// Global indices (ascending) of the variables in the dependency cone of centre unit i.
// RK4: unit i: 12 states + 4 inputs; units i+-1: 12 states + thrust; units i+-2: position + velocity.
// Euler: unit i: 12 + 4; units i+-1: position.
LEB_HD int window_vars(const Model& M, int i, int* vars /* >= 54 */) {
    int L = 0;
    const int U = M.n_units, n = M.n;
    const bool rk4 = (M.integ == 2);
    for (int q = i - 2; q <= i + 2; ++q) {
        if (q < 0 || q >= U) continue;
        int dq = q > i ? q - i : i - q;
        if (dq == 0) { for (int c = 0; c < 12; ++c) vars[L++] = 12 * q + c; }
        else if (dq == 1) {
            if (rk4) { for (int c = 0; c < 12; ++c) vars[L++] = 12 * q + c; }
            else { for (int c = 0; c < 3; ++c) vars[L++] = 12 * q + c; }
        } else if (rk4) {
            for (int c = 0; c < 3; ++c) vars[L++] = 12 * q + c;
            for (int c = 6; c < 9; ++c) vars[L++] = 12 * q + c;
        }
    }
    for (int q = i - 1; q <= i + 1; ++q) {
        if (q < 0 || q >= U) continue;
        if (q == i) { for (int c = 0; c < 4; ++c) vars[L++] = n + 4 * q + c; }
        else if (rk4) vars[L++] = n + 4 * q;
    }
    return L;
}

// off-diagonal item t in [0, L(L-1)/2) -> positions (a < b), row-major over a
LEB_HD void item_decode_offdiag(int t, int L, int* a, int* b) {
    int row = 0, rem = t;
    while (rem >= L - 1 - row) { rem -= L - 1 - row; ++row; }
    *a = row;
    *b = row + 1 + rem;
}

// item t in [0, L(L+1)/2) -> positions (a <= b) in the window list, row-major over a
LEB_HD void item_decode(int t, int L, int* a, int* b) {
    int row = 0, rem = t;
    while (rem >= L - row) { rem -= L - row; ++row; }
    *a = row;
    *b = row + rem;
}

// Contribution of item (j <= k) to R_l, eq. (15): off-diagonal [H_kj](A^(j)) D_j D_k, diagonal
// 1/2 [H_kk](A^(k)) sqr(D_k), D = [-sigma, sigma] (D_k^2 >= 0, L152).
template <class S>
LEB_HD Iv<S> item_term(const Iv<S>& H, const S& sj, const S& sk, bool diag) {
    if (diag) {
        Iv<S> Dk = {neg(sk), sk};
        return iscale(0.5f, imul(H, isqr(Dk)));
    }
    Iv<S> Dj = {neg(sj), sj}, Dk = {neg(sk), sk};
    return imul(H, imul(Dj, Dk));
}

}  // namespace leb_an

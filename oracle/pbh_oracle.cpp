// ORACLE (test infrastructure, NOT the product): path-based interval-Hessian (PBH)
// linearization-error bounds for analytic dynamics, plain FP64 C++17, one
// translation unit, no code shared with paper_2607_01203_b200/csrc.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference leg may load this library.
//
// What it follows (Sec. IV-A):
//   (10) L133      r(a; a~) = p(a) - p(a~) - J(a~)(a - a~)
//   (12) L147      R_classic = 1/2 D^T [H](A) D
//   (13) L152-155  R_expand  = sum_{j<k} [H_kj](A) D_j D_k + 1/2 sum_k [H_kk](A) D_k^2
//   (14) L157-162  prefix sets A^(k): coordinates > k pinned to the nominal point
//   (15) L164-167  R_path    = sum_{j<k} [H_kj](A^(j)) D_j D_k + 1/2 sum_k [H_kk](A^(k)) D_k^2
// with D = A (-) a~ (L164; L150 prints (+), a garble) and D_k^2 >= 0 (L152).
//
// The paper does not fix the inclusion function ("immrax", L236).  Reading R1
// (DESIGN.md): [H_l,kj](box) is the natural interval extension of second-order
// forward-mode AD of the model's straight-line program in directions (e_j, e_k);
// interval sin/cos are range-exact, interval * is min/max of the four endpoint
// products, sqr is non-negative.  The model SLPs (operation order included) are
// listed in DESIGN.md "Model SLPs" and restated below.
//
// VJP: forward-mode dual numbers through this same code, one pass per input
// direction; min/max select a branch by value, ties take the first candidate.
//
// Pins: tests/test_oracle_pbh.py (linear => 0, constant-Hessian closed form,
// unicycle closed form and hand-worked instance, Cor. 1 ordering (17), soundness
// against samples + all box vertices, central differences for the VJP).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ----------------------------------------------------------------- scalars
struct Dual { double v, d; };
inline double val(double x) { return x; }
inline double val(const Dual& x) { return x.v; }
inline double dot(double) { return 0.0; }
inline double dot(const Dual& x) { return x.d; }
template <class S> inline S cst(double c);
template <> inline double cst<double>(double c) { return c; }
template <> inline Dual cst<Dual>(double c) { return Dual{c, 0.0}; }

inline Dual operator+(Dual a, Dual b) { return {a.v + b.v, a.d + b.d}; }
inline Dual operator-(Dual a, Dual b) { return {a.v - b.v, a.d - b.d}; }
inline Dual operator-(Dual a) { return {-a.v, -a.d}; }
inline Dual operator*(Dual a, Dual b) { return {a.v * b.v, a.d * b.v + a.v * b.d}; }
inline Dual operator*(double c, Dual a) { return {c * a.v, c * a.d}; }
inline Dual operator/(Dual a, Dual b) { return {a.v / b.v, (a.d * b.v - a.v * b.d) / (b.v * b.v)}; }
inline double sin_(double x) { return std::sin(x); }
inline double cos_(double x) { return std::cos(x); }
inline Dual sin_(Dual x) { return {std::sin(x.v), std::cos(x.v) * x.d}; }
inline Dual cos_(Dual x) { return {std::cos(x.v), -std::sin(x.v) * x.d}; }
// branch selection by value; ties -> first argument
template <class S> inline S min_(S a, S b) { return val(b) < val(a) ? b : a; }
template <class S> inline S max_(S a, S b) { return val(b) > val(a) ? b : a; }

// ----------------------------------------------------------------- intervals
template <class S> struct Iv { S lo, hi; };
template <class S> inline Iv<S> ipoint(S x) { return {x, x}; }
template <class S> inline Iv<S> iconst(double c) { return {cst<S>(c), cst<S>(c)}; }
template <class S> inline bool is_zero(const Iv<S>& a) {
    return val(a.lo) == 0.0 && val(a.hi) == 0.0 && dot(a.lo) == 0.0 && dot(a.hi) == 0.0;
}
template <class S> inline Iv<S> operator+(Iv<S> a, Iv<S> b) { return {a.lo + b.lo, a.hi + b.hi}; }
template <class S> inline Iv<S> operator-(Iv<S> a, Iv<S> b) { return {a.lo - b.hi, a.hi - b.lo}; }
template <class S> inline Iv<S> operator-(Iv<S> a) { return {-a.hi, -a.lo}; }
template <class S> inline Iv<S> scale(double c, Iv<S> a) {
    if (c >= 0.0) return {c * a.lo, c * a.hi};
    return {c * a.hi, c * a.lo};
}
template <class S> inline Iv<S> operator*(Iv<S> a, Iv<S> b) {
    if (is_zero(a) || is_zero(b)) return iconst<S>(0.0);   // structural zero: result unchanged
    S p1 = a.lo * b.lo, p2 = a.lo * b.hi, p3 = a.hi * b.lo, p4 = a.hi * b.hi;
    return {min_(min_(min_(p1, p2), p3), p4), max_(max_(max_(p1, p2), p3), p4)};
}
template <class S> inline Iv<S> isqr(Iv<S> a) {
    if (val(a.lo) >= 0.0) return {a.lo * a.lo, a.hi * a.hi};
    if (val(a.hi) <= 0.0) return {a.hi * a.hi, a.lo * a.lo};
    return {cst<S>(0.0), max_(a.lo * a.lo, a.hi * a.hi)};
}
template <class S> inline Iv<S> icube(Iv<S> a) { return {a.lo * a.lo * a.lo, a.hi * a.hi * a.hi}; }
// range-exact sine / cosine
template <class S> inline Iv<S> isin(Iv<S> a) {
    const double PI = 3.14159265358979323846, TWO_PI = 2.0 * PI;
    double lo = val(a.lo), hi = val(a.hi);
    bool has_max, has_min;
    if (hi - lo >= TWO_PI) { has_max = has_min = true; }
    else {
        double kmax = std::ceil((lo - 0.5 * PI) / TWO_PI);
        has_max = (0.5 * PI + TWO_PI * kmax) <= hi;
        double kmin = std::ceil((lo + 0.5 * PI) / TWO_PI);
        has_min = (-0.5 * PI + TWO_PI * kmin) <= hi;
    }
    S sl = sin_(a.lo), sh = sin_(a.hi);
    Iv<S> r;
    r.hi = has_max ? cst<S>(1.0) : max_(sl, sh);
    r.lo = has_min ? cst<S>(-1.0) : min_(sl, sh);
    return r;
}
template <class S> inline Iv<S> icos(Iv<S> a) {
    const double PI = 3.14159265358979323846, TWO_PI = 2.0 * PI;
    double lo = val(a.lo), hi = val(a.hi);
    bool has_max, has_min;
    if (hi - lo >= TWO_PI) { has_max = has_min = true; }
    else {
        double kmax = std::ceil(lo / TWO_PI);
        has_max = (TWO_PI * kmax) <= hi;
        double kmin = std::ceil((lo - PI) / TWO_PI);
        has_min = (PI + TWO_PI * kmin) <= hi;
    }
    S cl = cos_(a.lo), ch = cos_(a.hi);
    Iv<S> r;
    r.hi = has_max ? cst<S>(1.0) : max_(cl, ch);
    r.lo = has_min ? cst<S>(-1.0) : min_(cl, ch);
    return r;
}
struct DomainError {};
template <class S> inline Iv<S> irecip(Iv<S> a) {
    if (val(a.lo) <= 0.0 && val(a.hi) >= 0.0) throw DomainError{};
    return {cst<S>(1.0) / a.hi, cst<S>(1.0) / a.lo};
}

// ----------------------------------------------------------------- second-order jets
// (w, w_j, w_k, w_jk) of reading R1; `diag` marks j == k.
template <class S> struct Jet {
    Iv<S> w, wj, wk, wjk;
    bool diag;
};
template <class S> inline Jet<S> jconst(double c, bool diag) {
    return {iconst<S>(c), iconst<S>(0.0), iconst<S>(0.0), iconst<S>(0.0), diag};
}
template <class S> inline Jet<S> operator+(const Jet<S>& a, const Jet<S>& b) {
    return {a.w + b.w, a.wj + b.wj, a.wk + b.wk, a.wjk + b.wjk, a.diag};
}
template <class S> inline Jet<S> operator-(const Jet<S>& a, const Jet<S>& b) {
    return {a.w - b.w, a.wj - b.wj, a.wk - b.wk, a.wjk - b.wjk, a.diag};
}
template <class S> inline Jet<S> operator-(const Jet<S>& a) { return {-a.w, -a.wj, -a.wk, -a.wjk, a.diag}; }
template <class S> inline Jet<S> scale(double c, const Jet<S>& a) {
    return {scale(c, a.w), scale(c, a.wj), scale(c, a.wk), scale(c, a.wjk), a.diag};
}
template <class S> inline Jet<S> addc(const Jet<S>& a, double c) {
    Jet<S> r = a;
    r.w = a.w + iconst<S>(c);
    return r;
}
template <class S> inline Jet<S> operator*(const Jet<S>& a, const Jet<S>& b) {
    Jet<S> r;
    r.diag = a.diag;
    r.w = a.w * b.w;
    r.wj = a.wj * b.w + a.w * b.wj;
    r.wk = a.wk * b.w + a.w * b.wk;
    Iv<S> cross = a.diag ? scale(2.0, a.wj * b.wj) : (a.wj * b.wk + a.wk * b.wj);
    r.wjk = a.wjk * b.w + cross + a.w * b.wjk;
    return r;
}
// unary w = phi(a) given enclosures of phi(a), phi'(a), phi''(a)
template <class S> inline Jet<S> unary(const Jet<S>& a, Iv<S> f, Iv<S> f1, Iv<S> f2) {
    Jet<S> r;
    r.diag = a.diag;
    r.w = f;
    r.wj = f1 * a.wj;
    r.wk = f1 * a.wk;
    Iv<S> jk = a.diag ? isqr(a.wj) : (a.wj * a.wk);
    r.wjk = f2 * jk + f1 * a.wjk;
    return r;
}
template <class S> inline Jet<S> sin_(const Jet<S>& a) { Iv<S> s = isin(a.w), c = icos(a.w); return unary(a, s, c, -s); }
template <class S> inline Jet<S> cos_(const Jet<S>& a) { Iv<S> s = isin(a.w), c = icos(a.w); return unary(a, c, -s, -c); }
template <class S> inline Jet<S> recip_(const Jet<S>& a) {
    Iv<S> r = irecip(a.w);
    return unary(a, r, -isqr(r), scale(2.0, icube(r)));
}
template <class S> inline Jet<S> sqr_(const Jet<S>& a) { return unary(a, isqr(a.w), scale(2.0, a.w), iconst<S>(2.0)); }
template <class S> inline Jet<S> cube_(const Jet<S>& a) { return unary(a, icube(a.w), scale(3.0, isqr(a.w)), scale(6.0, a.w)); }

// plain-double versions of the same primitives, so the model SLPs below can also
// be evaluated pointwise (true f for sampling tests)
inline double scale(double c, double a) { return c * a; }
inline double addc(double a, double c) { return a + c; }
inline double recip_(double a) { return 1.0 / a; }
inline double sqr_(double a) { return a * a; }
inline double cube_(double a) { return a * a * a; }

// ----------------------------------------------------------------- models
struct Params { double dt, mass, g, Jx, Jy, Jz, k1, k3; };
enum { MODEL_UNICYCLE = 1, MODEL_QUAD12 = 2, MODEL_QUADCHAIN = 3, MODEL_PLANAR_QUAD = 4, MODEL_SATELLITE = 5,
       MODEL_QUADCENTROID = 6,
       MODEL_QUADRATIC = 100, MODEL_LINEAR = 101 };
enum { INTEG_EULER = 1, INTEG_RK4 = 2 };

// quad12 vector field g(xi, nu), DESIGN.md "Model SLPs" (state order PAPER.md:L538;
// eq. (38a) L534 is garbled, the standard ZYX form is used -- reading R6).
// xi = (px,py,pz, phi,theta,psi, vx,vy,vz, p,q,r), nu = (T, tau_phi, tau_theta, tau_psi).
// `coup` = coupling force per axis (already summed), added as (1/m)*coup.
template <class X>
void quad12_field(const Params& P, const X* xi, const X* nu, const X* coup, X* out) {
    const X &phi = xi[3], &th = xi[4], &psi = xi[5];
    const X &p = xi[9], &q = xi[10], &r = xi[11];
    X sphi = sin_(phi), cphi = cos_(phi), sth = sin_(th), cth = cos_(th), spsi = sin_(psi), cpsi = cos_(psi);
    X rcth = recip_(cth);
    X a = q * sphi + r * cphi;
    out[0] = xi[6];
    out[1] = xi[7];
    out[2] = xi[8];
    out[3] = p + a * (sth * rcth);
    out[4] = q * cphi - r * sphi;
    out[5] = a * rcth;
    X Tm = scale(1.0 / P.mass, nu[0]);
    out[6] = Tm * ((cpsi * sth) * cphi + spsi * sphi);
    out[7] = Tm * ((spsi * sth) * cphi - cpsi * sphi);
    out[8] = addc(Tm * (cth * cphi), -P.g);
    out[9] = scale((P.Jy - P.Jz) / P.Jx, q * r) + scale(1.0 / P.Jx, nu[1]);
    out[10] = scale((P.Jz - P.Jx) / P.Jy, p * r) + scale(1.0 / P.Jy, nu[2]);
    out[11] = scale((P.Jx - P.Jy) / P.Jz, p * q) + scale(1.0 / P.Jz, nu[3]);
    if (coup) {
        for (int c = 0; c < 3; ++c) out[6 + c] = out[6 + c] + scale(1.0 / P.mass, coup[c]);
    }
}

// chain vector field: U units; spring i joins units i and i+1, per axis c:
//   d = p_{i+1,c} - p_{i,c},  s = k1*d + k3*cube(d);  force on i: +s, on i+1: -s.
template <class X>
void chain_field(const Params& P, int U, const X* x, const X* u, X* out) {
    std::vector<X> s(3 * std::max(U - 1, 1), x[0]);
    for (int i = 0; i + 1 < U; ++i)
        for (int c = 0; c < 3; ++c) {
            X d = x[12 * (i + 1) + c] - x[12 * i + c];
            s[3 * i + c] = scale(P.k1, d) + scale(P.k3, cube_(d));
        }
    for (int i = 0; i < U; ++i) {
        X coup[3] = {x[0], x[0], x[0]};
        bool any = false;
        for (int c = 0; c < 3; ++c) {
            if (i + 1 < U && i > 0) { coup[c] = s[3 * i + c] - s[3 * (i - 1) + c]; any = true; }
            else if (i + 1 < U) { coup[c] = s[3 * i + c]; any = true; }
            else if (i > 0) { coup[c] = -s[3 * (i - 1) + c]; any = true; }
        }
        quad12_field(P, x + 12 * i, u + 4 * i, any ? coup : (const X*)nullptr, out + 12 * i);
    }
}

// coupled 3-D quadrotors of the paper, eq. (39)-(42) PAPER.md:L540-558: U quad12 units, centroid spring-damper
//   a_i = -alpha U (p_i - pbar) - gamma (v_i - vbar),  pbar = (1/U) sum p_i,  vbar = (1/U) sum v_i        (40)-(41)
// added to the translational acceleration of unit i (42).  Params: k1 = alpha, k3 = gamma.
template <class X>
void centroid_field(const Params& P, int U, const X* x, const X* u, X* out) {
    X pbar[3] = {x[0], x[0], x[0]}, vbar[3] = {x[0], x[0], x[0]};
    for (int c = 0; c < 3; ++c) {
        X sp = x[c], sv = x[6 + c];
        for (int i = 1; i < U; ++i) { sp = sp + x[12 * i + c]; sv = sv + x[12 * i + 6 + c]; }
        pbar[c] = scale(1.0 / U, sp);
        vbar[c] = scale(1.0 / U, sv);
    }
    for (int i = 0; i < U; ++i) {
        quad12_field(P, x + 12 * i, u + 4 * i, (const X*)nullptr, out + 12 * i);
        for (int c = 0; c < 3; ++c) {
            X a = scale(-P.k1 * U, x[12 * i + c] - pbar[c]) + scale(-P.k3, x[12 * i + 6 + c] - vbar[c]);
            out[12 * i + 6 + c] = out[12 * i + 6 + c] + a;
        }
    }
}

// planar quadrotor, eq. (37a): x = (px, py, phi, vx, vy, phidot), u = (u1, u2);
// xdot = (vx, vy, phidot, -(u1+u2) sin(phi)/m, (u1+u2) cos(phi)/m - g, (L/J)(u2 - u1))   ("L/T" at L524 is a garble of L/J).
// Params: mass = m, g, Jx = J, k1 = L.
template <class X>
void planar_quad_field(const Params& P, const X* x, const X* u, X* out) {
    X s = sin_(x[2]), c = cos_(x[2]);
    X thrust = scale(1.0 / P.mass, u[0] + u[1]);
    out[0] = x[3];
    out[1] = x[4];
    out[2] = x[5];
    out[3] = -(thrust * s);
    out[4] = addc(thrust * c, -P.g);
    out[5] = scale(P.k1 / P.Jx, u[1] - u[0]);
}

// satellite, eq. (36): x = (q[4], om[3]), u = torque[3];
// qdot = zeta(om) q (the 4x4 matrix printed at L514), omdot = I^-1 (u - om x (I om)), I = diag(Jx, Jy, Jz).
template <class X>
void satellite_field(const Params& P, const X* x, const X* u, X* out) {
    const X* q = x;
    const X* om = x + 4;
    out[0] = scale(0.5, ((-(om[0] * q[1])) - om[1] * q[2]) - om[2] * q[3]);
    out[1] = scale(0.5, (om[0] * q[0] + om[2] * q[2]) - om[1] * q[3]);
    out[2] = scale(0.5, (om[1] * q[0] - om[2] * q[1]) + om[0] * q[3]);
    out[3] = scale(0.5, (om[2] * q[0] + om[1] * q[1]) - om[0] * q[2]);
    // (om x I om) = ((Jz - Jy) om2 om3, (Jx - Jz) om3 om1, (Jy - Jx) om1 om2)
    out[4] = scale((P.Jy - P.Jz) / P.Jx, om[1] * om[2]) + scale(1.0 / P.Jx, u[0]);
    out[5] = scale((P.Jz - P.Jx) / P.Jy, om[0] * om[2]) + scale(1.0 / P.Jy, u[1]);
    out[6] = scale((P.Jx - P.Jy) / P.Jz, om[0] * om[1]) + scale(1.0 / P.Jz, u[2]);
}

struct Model {
    int id, integ, n_units;
    Params P;
    const double* Q;   // MODEL_QUADRATIC: n x N x N, f_l = 1/2 a^T Q_l a + c_l^T a ; MODEL_LINEAR: n x N
    const double* C;
    int n, N;
};

template <class X>
void vector_field(const Model& M, const X* x, const X* u, X* out) {
    if (M.id == MODEL_QUAD12) quad12_field<X>(M.P, x, u, nullptr, out);
    else if (M.id == MODEL_PLANAR_QUAD) planar_quad_field<X>(M.P, x, u, out);
    else if (M.id == MODEL_SATELLITE) satellite_field<X>(M.P, x, u, out);
    else if (M.id == MODEL_QUADCENTROID) centroid_field<X>(M.P, M.n_units, x, u, out);
    else chain_field<X>(M.P, M.n_units, x, u, out);
}

// discrete-time map f(alpha), alpha = [x; u]
template <class X>
void model_f(const Model& M, const X* al, X* f) {
    const int n = M.n, N = M.N;
    if (M.id == MODEL_UNICYCLE) {
        // f = (px + dt*(v*cos th), py + dt*(v*sin th), th + dt*om);  alpha = (px,py,th,v,om)
        f[0] = al[0] + scale(M.P.dt, al[3] * cos_(al[2]));
        f[1] = al[1] + scale(M.P.dt, al[3] * sin_(al[2]));
        f[2] = al[2] + scale(M.P.dt, al[4]);
        return;
    }
    if (M.id == MODEL_LINEAR) {
        for (int l = 0; l < n; ++l) {
            X acc = scale(M.C[l * N], al[0]);
            for (int i = 1; i < N; ++i) acc = acc + scale(M.C[l * N + i], al[i]);
            f[l] = acc;
        }
        return;
    }
    if (M.id == MODEL_QUADRATIC) {
        for (int l = 0; l < n; ++l) {
            X acc = scale(M.C[l * N], al[0]);
            for (int i = 1; i < N; ++i) acc = acc + scale(M.C[l * N + i], al[i]);
            for (int i = 0; i < N; ++i)
                for (int k = 0; k < N; ++k) {
                    double qv = M.Q[(l * N + i) * N + k];
                    if (qv != 0.0) acc = acc + scale(0.5 * qv, al[i] * al[k]);
                }
            f[l] = acc;
        }
        return;
    }
    const X* x = al;
    const X* u = al + n;
    const double dt = M.P.dt;
    std::vector<X> k1(n, al[0]), k2(n, al[0]), k3(n, al[0]), k4(n, al[0]), xs(n, al[0]);
    vector_field(M, x, u, k1.data());
    if (M.integ == INTEG_EULER) {
        for (int i = 0; i < n; ++i) f[i] = x[i] + scale(dt, k1[i]);
        return;
    }
    for (int i = 0; i < n; ++i) xs[i] = x[i] + scale(0.5 * dt, k1[i]);
    vector_field(M, xs.data(), u, k2.data());
    for (int i = 0; i < n; ++i) xs[i] = x[i] + scale(0.5 * dt, k2[i]);
    vector_field(M, xs.data(), u, k3.data());
    for (int i = 0; i < n; ++i) xs[i] = x[i] + scale(dt, k3[i]);
    vector_field(M, xs.data(), u, k4.data());
    for (int i = 0; i < n; ++i)
        f[i] = x[i] + scale(dt / 6.0, ((k1[i] + scale(2.0, k2[i])) + scale(2.0, k3[i])) + k4[i]);
}

// ----------------------------------------------------------------- PBH, eq. (12)/(13)/(15)
enum { MODE_PATH = 0, MODE_EXPAND = 1, MODE_CLASSIC = 2 };

// [H_{l,kj}](box) for all outputs l: second-order jets in directions (e_j, e_k).
// box[i] is an interval for i in the "interval" set, a point otherwise.
template <class S>
void hessian_entry(const Model& M, const std::vector<Iv<S>>& box, int j, int k, std::vector<Iv<S>>& H) {
    const int N = M.N, n = M.n;
    const bool diag = (j == k);
    std::vector<Jet<S>> al(N), f(n);
    for (int i = 0; i < N; ++i) {
        al[i].w = box[i];
        al[i].wj = iconst<S>(i == j ? 1.0 : 0.0);
        al[i].wk = iconst<S>(i == k ? 1.0 : 0.0);
        al[i].wjk = iconst<S>(0.0);
        al[i].diag = diag;
    }
    model_f<Jet<S>>(M, al.data(), f.data());
    for (int l = 0; l < n; ++l) H[l] = f[l].wjk;
}

// one tile.  nom, rad, mu: N scalars (S carries tangents for the VJP); mu may be NULL (= 0).
//
// Non-centred boxes (25a) L272: A_i = (a~_i + mu_i) + [-sigma_i, sigma_i], so Delta_i = A_i (-) a~_i =
// [mu_i - sigma_i, mu_i + sigma_i] (L164).  Thm 1 needs a~ in the set the Hessian is enclosed on (L164: the path
// runs from a~ to a point of A one coordinate at a time), which (25a) does not give when |mu_i| > sigma_i; reading
// R4: the enclosure is taken on hull(A_i u {a~_i}) = a~_i + [min(mu_i - sigma_i, 0), max(mu_i + sigma_i, 0)]
// -- every point of the segment from a~_i to a point of A_i.  With mu = 0 this is A_i itself.
template <class S>
void pbh_tile(const Model& M, const S* nom, const S* rad, const S* mu, int mode, S* r_lo, S* r_hi) {
    const int N = M.N, n = M.n;
    std::vector<Iv<S>> A(N), D(N), box(N), H(n);
    for (int i = 0; i < N; ++i) {
        if (mu) {
            D[i] = {mu[i] - rad[i], mu[i] + rad[i]};        // Delta = A (-) a~
            // ties keep the first candidate (the VJP then follows mu -+ sigma)
            A[i] = {nom[i] + min_(D[i].lo, cst<S>(0.0)), nom[i] + max_(D[i].hi, cst<S>(0.0))};
        } else {
            A[i] = {nom[i] - rad[i], nom[i] + rad[i]};      // (25a) with mu = 0
            D[i] = {-rad[i], rad[i]};                       // Delta = A (-) a~
        }
    }
    std::vector<Iv<S>> R(n, iconst<S>(0.0));
    if (mode == MODE_CLASSIC) {
        // (12): 1/2 sum_j sum_k [H_jk](A) D_j D_k, plain interval products
        for (int j = 0; j < N; ++j)
            for (int k = 0; k < N; ++k) {
                hessian_entry<S>(M, A, std::min(j, k), std::max(j, k), H);
                for (int l = 0; l < n; ++l) R[l] = R[l] + scale(0.5, H[l] * (D[j] * D[k]));
            }
    } else {
        for (int j = 0; j < N; ++j) {
            // prefix box A^(j) (14): coordinates <= j interval, > j pinned to the nominal
            for (int i = 0; i < N; ++i)
                box[i] = (mode == MODE_EXPAND || i <= j) ? A[i] : ipoint<S>(nom[i]);
            for (int k = j; k < N; ++k) {
                hessian_entry<S>(M, box, j, k, H);
                if (k == j) {
                    Iv<S> d2 = isqr(D[k]);                  // Delta_k^2 >= 0  (L152)
                    for (int l = 0; l < n; ++l) R[l] = R[l] + scale(0.5, H[l] * d2);
                } else {
                    Iv<S> dd = D[j] * D[k];
                    for (int l = 0; l < n; ++l) R[l] = R[l] + H[l] * dd;
                }
            }
        }
    }
    for (int l = 0; l < n; ++l) { r_lo[l] = R[l].lo; r_hi[l] = R[l].hi; }
}

Model make_model(int id, int integ, int n_units, const double* params, const double* Q, const double* C, int n, int N) {
    Model M;
    M.id = id; M.integ = integ; M.n_units = n_units;
    M.P = Params{params[0], params[1], params[2], params[3], params[4], params[5], params[6], params[7]};
    M.Q = Q; M.C = C;
    if (id == MODEL_UNICYCLE) { M.n = 3; M.N = 5; }
    else if (id == MODEL_QUAD12) { M.n = 12; M.N = 16; }
    else if (id == MODEL_QUADCHAIN || id == MODEL_QUADCENTROID) { M.n = 12 * n_units; M.N = 16 * n_units; }
    else if (id == MODEL_PLANAR_QUAD) { M.n = 6; M.N = 8; }
    else if (id == MODEL_SATELLITE) { M.n = 7; M.N = 10; }
    else { M.n = n; M.N = N; }
    return M;
}

}  // namespace

extern "C" {

// status: 0 ok, 4 domain error (0 in cos(theta) box) in some tile -> that tile's bounds are -/+inf
int pbh_oracle_eval(int model_id, int integ, int n_units, const double* params,
                    const double* Q, const double* C, int n_gen, int N_gen,
                    int tiles, const double* nom, const double* rad, const double* mu, int mode,
                    double* r_lo, double* r_hi, int threads) {
    Model M = make_model(model_id, integ, n_units, params, Q, C, n_gen, N_gen);
    int status = 0;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int t = 0; t < tiles; ++t) {
        try {
            pbh_tile<double>(M, nom + (size_t)t * M.N, rad + (size_t)t * M.N, mu ? mu + (size_t)t * M.N : nullptr, mode,
                             r_lo + (size_t)t * M.n, r_hi + (size_t)t * M.n);
        } catch (DomainError&) {
            for (int l = 0; l < M.n; ++l) { r_lo[(size_t)t * M.n + l] = -INFINITY; r_hi[(size_t)t * M.n + l] = INFINITY; }
#pragma omp critical
            status = 4;
        }
    }
    return status;
}

// VJP by forward-mode duals.  dirs: list of n_dirs direction indices in [0, 3N):
// d < N -> d/d nom[d], N <= d < 2N -> d/d rad[d-N], d >= 2N -> d/d mu[d-2N] (mu != NULL only).
// out[t*n_dirs + i] =
// sum_l g_hi[l] d r_hi[l] + g_lo[l] d r_lo[l]  along direction dirs[i].
int pbh_oracle_vjp(int model_id, int integ, int n_units, const double* params,
                   const double* Q, const double* C, int n_gen, int N_gen,
                   int tiles, const double* nom, const double* rad, const double* mu,
                   const double* g_lo, const double* g_hi,
                   int n_dirs, const int* dirs, double* out, int threads) {
    Model M = make_model(model_id, integ, n_units, params, Q, C, n_gen, N_gen);
    const int N = M.N, n = M.n;
    int status = 0;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
    for (int t = 0; t < tiles; ++t)
        for (int i = 0; i < n_dirs; ++i) {
            std::vector<Dual> a(N), s(N), m(N), lo(n), hi(n);
            const int d = dirs[i];
            for (int q = 0; q < N; ++q) {
                a[q] = Dual{nom[(size_t)t * N + q], (d == q) ? 1.0 : 0.0};
                s[q] = Dual{rad[(size_t)t * N + q], (d == N + q) ? 1.0 : 0.0};
                m[q] = Dual{mu ? mu[(size_t)t * N + q] : 0.0, (d == 2 * N + q) ? 1.0 : 0.0};
            }
            try {
                pbh_tile<Dual>(M, a.data(), s.data(), mu ? m.data() : nullptr, MODE_PATH, lo.data(), hi.data());
                double acc = 0.0;
                for (int l = 0; l < n; ++l)
                    acc += g_hi[(size_t)t * n + l] * hi[l].d + g_lo[(size_t)t * n + l] * lo[l].d;
                out[(size_t)t * n_dirs + i] = acc;
            } catch (DomainError&) {
                out[(size_t)t * n_dirs + i] = NAN;
#pragma omp critical
                status = 4;
            }
        }
    return status;
}

// pointwise f(alpha) (true function, for sampling tests): pts x N -> pts x n
void pbh_oracle_f(int model_id, int integ, int n_units, const double* params,
                  const double* Q, const double* C, int n_gen, int N_gen,
                  int pts, const double* alpha, double* f) {
    Model M = make_model(model_id, integ, n_units, params, Q, C, n_gen, N_gen);
#pragma omp parallel for
    for (int t = 0; t < pts; ++t) model_f<double>(M, alpha + (size_t)t * M.N, f + (size_t)t * M.n);
}

// Jacobian J(alpha) = [A_k B_k] (7) at one point, from first-order jet parts at a point box: n x N
void pbh_oracle_jac(int model_id, int integ, int n_units, const double* params,
                    const double* Q, const double* C, int n_gen, int N_gen,
                    const double* alpha, double* J) {
    Model M = make_model(model_id, integ, n_units, params, Q, C, n_gen, N_gen);
    const int N = M.N, n = M.n;
    for (int j = 0; j < N; ++j) {
        std::vector<Jet<double>> al(N), f(n);
        for (int i = 0; i < N; ++i) {
            al[i].w = ipoint<double>(alpha[i]);
            al[i].wj = iconst<double>(i == j ? 1.0 : 0.0);
            al[i].wk = iconst<double>(0.0);
            al[i].wjk = iconst<double>(0.0);
            al[i].diag = false;
        }
        model_f<Jet<double>>(M, al.data(), f.data());
        for (int l = 0; l < n; ++l) J[l * N + j] = f[l].wj.lo;
    }
}

// one Hessian column enclosure (tests): H[l] = [H_{l,kj}](box) with box given as lo/hi arrays
void pbh_oracle_hessian_entry(int model_id, int integ, int n_units, const double* params,
                              const double* Q, const double* C, int n_gen, int N_gen,
                              const double* box_lo, const double* box_hi, int j, int k,
                              double* H_lo, double* H_hi) {
    Model M = make_model(model_id, integ, n_units, params, Q, C, n_gen, N_gen);
    std::vector<Iv<double>> box(M.N), H(M.n);
    for (int i = 0; i < M.N; ++i) box[i] = {box_lo[i], box_hi[i]};
    hessian_entry<double>(M, box, j, k, H);
    for (int l = 0; l < M.n; ++l) { H_lo[l] = H[l].lo; H_hi[l] = H[l].hi; }
}

int pbh_oracle_max_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"

// an_compile.cu -- host side of the analytic path: symbolic evaluation of a model's straight-line program
// (SLP) into the interval tape of an_tape.h.  Structure only -- no interval is evaluated here; every number
// of the bound is computed by the device interpreter (analytic.cu).
//
// For every path index j (eq. (14)-(15)) the model SLP is run on symbolic second-order
// jets (reading R1): a component is `zero`, a constant c (the seeds e_j, e_k are the constant 1), or a slot
// of the tape.  0 * x = 0, 0 + x = x, 1 * x = x and c * [lo, hi] = the hull of the endpoint products are exact
// identities of the interval extension (also under directed rounding), so dropping / folding them leaves
// the enclosure the contract defines; two constants are folded only when the FP32 result is exact.
//   pass WJ(j)   : w and w_j of every SLP variable on the prefix box A^(j); results memoised in evaluation order
//   pass K(j,k)  : the same SLP again for every k >= j that shares an output with j; w and w_j come from the
//                  memo (the SLP is straight-line: the sequence of operations is the same), w_k and w_jk are new
// then dead code is removed (backwards from the OUT instructions) and slots are renumbered.
#include <math.h>
#include <string.h>
#include <algorithm>
#include <unordered_map>
#include "an_tape.h"
#include "internal.h"

namespace leb_an {
namespace {

enum SK : uint8_t { SK_Z = 0, SK_C = 1, SK_S = 2 };
struct Sym {
    SK k = SK_Z;
    float c = 0.f;     // SK_C
    uint32_t s = 0;    // SK_S: slot id; bit 30 set = slot of the current K segment, else of WJ
};
constexpr uint32_t KTAG = 1u << 30;

inline Sym Z() { return Sym{}; }
inline Sym C(float c) { Sym r; if (c == 0.f) return r; r.k = SK_C; r.c = c; return r; }
inline Sym S(uint32_t s) { Sym r; r.k = SK_S; r.s = s; return r; }
inline uint32_t fbits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }
inline bool exact_f32(double v) { return (double)(float)v == v && fabs(v) < 3.0e38; }

struct SJet { Sym w, wj, wk, wjk; };

class Builder {
public:
    // ---- emission state
    std::vector<Ins> wj_ins, k_ins;
    bool kphase = false, diag = false;
    std::vector<Sym> memo;
    size_t mpos = 0;
    std::unordered_map<uint32_t, uint32_t> const_wj, const_k;     // float bits -> slot
    int j = 0, k = 0;
    bool use_mu = false;
    std::vector<int> in_slot;        // input coordinate -> slot of its w in WJ (or -1)

    uint32_t emit(uint32_t op, uint32_t a, uint32_t b) {
        std::vector<Ins>& v = kphase ? k_ins : wj_ins;
        uint32_t slot = (uint32_t)v.size() | (kphase ? KTAG : 0u);
        // an operand slot is stored with its tag; resolved to a final index when the task is laid out
        v.push_back(Ins{op, a});      // temporarily: w0 = op, w1 = a ; b kept in the side array
        (kphase ? k_b : wj_b).push_back(b);
        return slot;
    }
    std::vector<uint32_t> wj_b, k_b;

    Sym mat(Sym a) {                 // constants become slots when an instruction needs one
        if (a.k != SK_C) return a;
        auto& cache = kphase ? const_k : const_wj;
        auto it = cache.find(fbits(a.c));
        if (it != cache.end()) return S(it->second);
        // a constant needed in a K segment may already exist in WJ
        if (kphase) { auto iw = const_wj.find(fbits(a.c)); if (iw != const_wj.end()) return S(iw->second); }
        uint32_t s = emit(OP_CONST, 0, fbits(a.c));
        cache[fbits(a.c)] = s;
        return S(s);
    }
    Sym un(uint32_t op, Sym a) { a = mat(a); return S(emit(op, a.s, 0)); }
    Sym neg(Sym a) {
        if (a.k == SK_Z) return a;
        if (a.k == SK_C) return C(-a.c);
        return S(emit(OP_NEG, a.s, 0));
    }
    Sym scale(float c, Sym a) {
        if (c == 0.f || a.k == SK_Z) return Z();
        if (c == 1.f) return a;
        if (a.k == SK_C) {
            double p = (double)c * (double)a.c;
            if (exact_f32(p)) return C((float)p);
            a = mat(a);
        }
        return S(emit(OP_SCALE, a.s, fbits(c)));
    }
    Sym addc(Sym a, float c) {
        if (c == 0.f) return a;
        if (a.k == SK_Z) return C(c);
        if (a.k == SK_C) {
            double s = (double)a.c + (double)c;
            if (exact_f32(s)) return C((float)s);
            a = mat(a);
        }
        return S(emit(OP_ADDC, a.s, fbits(c)));
    }
    Sym add(Sym a, Sym b) {
        if (a.k == SK_Z) return b;
        if (b.k == SK_Z) return a;
        if (a.k == SK_C && b.k == SK_C) {
            double s = (double)a.c + (double)b.c;
            if (exact_f32(s)) return C((float)s);
            a = mat(a);
        }
        if (a.k == SK_C) return addc(b, a.c);
        if (b.k == SK_C) return addc(a, b.c);
        return S(emit(OP_ADD, a.s, b.s));
    }
    Sym sub(Sym a, Sym b) {
        if (b.k == SK_Z) return a;
        if (a.k == SK_Z) return neg(b);
        if (b.k == SK_C) return add(a, C(-b.c));
        if (a.k == SK_C) return addc(neg(b), a.c);
        return S(emit(OP_SUB, a.s, b.s));
    }
    Sym mul(Sym a, Sym b) {
        if (a.k == SK_Z || b.k == SK_Z) return Z();
        if (a.k == SK_C) return scale(a.c, b);
        if (b.k == SK_C) return scale(b.c, a);
        return S(emit(OP_MUL, a.s, b.s));
    }
    Sym sqr(Sym a) {
        if (a.k == SK_Z) return a;
        if (a.k == SK_C) {
            double p = (double)a.c * (double)a.c;
            if (exact_f32(p)) return C((float)p);
            a = mat(a);
        }
        return S(emit(OP_SQR, a.s, 0));
    }

    // w / w_j components: computed in pass WJ, replayed from the memo in pass K
    template <class F> Sym M(F&& f) {
        if (kphase) return memo[mpos++];
        Sym r = f();
        memo.push_back(r);
        return r;
    }

    // ---- inputs: prefix box A^(j) (14) L157-162
    SJet in(int g) {
        SJet r;
        r.w = M([&] {
            if (in_slot[g] < 0) {
                uint32_t op = g <= j ? (use_mu ? OP_BOXMU : OP_BOX) : OP_PT;
                in_slot[g] = (int)emit(op, (uint32_t)g, 0);
            }
            return S((uint32_t)in_slot[g]);
        });
        r.wj = g == j ? C(1.f) : Z();
        r.wk = g == k ? C(1.f) : Z();
        r.wjk = Z();
        return r;
    }
    SJet cst(float c) { SJet r; r.w = C(c); return r; }

    // ---- jet arithmetic (reading R1)
    SJet jadd(const SJet& a, const SJet& b) {
        SJet r;
        r.w = M([&] { return add(a.w, b.w); });
        r.wj = M([&] { return add(a.wj, b.wj); });
        if (kphase) { r.wk = diag ? r.wj : add(a.wk, b.wk); r.wjk = add(a.wjk, b.wjk); }
        return r;
    }
    SJet jsub(const SJet& a, const SJet& b) {
        SJet r;
        r.w = M([&] { return sub(a.w, b.w); });
        r.wj = M([&] { return sub(a.wj, b.wj); });
        if (kphase) { r.wk = diag ? r.wj : sub(a.wk, b.wk); r.wjk = sub(a.wjk, b.wjk); }
        return r;
    }
    SJet jneg(const SJet& a) {
        SJet r;
        r.w = M([&] { return neg(a.w); });
        r.wj = M([&] { return neg(a.wj); });
        if (kphase) { r.wk = diag ? r.wj : neg(a.wk); r.wjk = neg(a.wjk); }
        return r;
    }
    SJet jscale(float c, const SJet& a) {
        SJet r;
        r.w = M([&] { return scale(c, a.w); });
        r.wj = M([&] { return scale(c, a.wj); });
        if (kphase) { r.wk = diag ? r.wj : scale(c, a.wk); r.wjk = scale(c, a.wjk); }
        return r;
    }
    SJet jaddc(const SJet& a, float c) {
        SJet r = a;
        r.w = M([&] { return addc(a.w, c); });
        return r;
    }
    // product rule; on the diagonal (j == k) the cross term is 2 a_j b_j
    SJet jmul(const SJet& a, const SJet& b) {
        SJet r;
        r.w = M([&] { return mul(a.w, b.w); });
        // sums are emitted as running sums (t; m; t + m) so that the peephole can fuse each product into its addition
        r.wj = M([&] { Sym t = mul(a.wj, b.w); return add(t, mul(a.w, b.wj)); });
        if (kphase) {
            if (diag) r.wk = r.wj;
            else { Sym t = mul(a.wk, b.w); r.wk = add(t, mul(a.w, b.wk)); }
            Sym t;
            if (diag) t = scale(2.f, mul(a.wj, b.wj));
            else { t = mul(a.wj, b.wk); t = add(t, mul(a.wk, b.wj)); }
            t = add(t, mul(a.wjk, b.w));
            r.wjk = add(t, mul(a.w, b.wjk));
        }
        return r;
    }
    // w = phi(a) from enclosures f, f1, f2 of phi, phi', phi'' on a.w; on the diagonal a_j a_k = sqr(a_j)
    SJet junary(const SJet& a, Sym f, Sym f1, Sym f2) {
        SJet r;
        r.w = f;
        r.wj = M([&] { return mul(f1, a.wj); });
        if (kphase) {
            r.wk = diag ? r.wj : mul(f1, a.wk);
            Sym jk = diag ? sqr(a.wj) : mul(a.wj, a.wk);
            Sym t = mul(f2, jk);
            r.wjk = add(t, mul(f1, a.wjk));
        }
        return r;
    }
    void jsincos(const SJet& a, SJet* s_out, SJet* c_out) {
        Sym s = M([&] { return un(OP_SIN, a.w); });
        Sym c = M([&] { return un(OP_COS, a.w); });
        Sym ns = M([&] { return neg(s); });
        Sym nc = M([&] { return neg(c); });
        *s_out = junary(a, s, c, ns);        // (sin)' = cos, (sin)'' = -sin
        *c_out = junary(a, c, ns, nc);       // (cos)' = -sin, (cos)'' = -cos
    }
    SJet jrecip(const SJet& a) {
        Sym r = M([&] { return un(OP_RECIP, a.w); });
        Sym f1 = M([&] { return neg(sqr(r)); });                     // (1/a)' = -1/a^2
        Sym f2 = M([&] { return scale(2.f, un(OP_CUBE, r)); });      // (1/a)'' = 2/a^3
        return junary(a, r, f1, f2);
    }
    SJet jcube(const SJet& a) {
        Sym f = M([&] { return un(OP_CUBE, a.w); });
        Sym f1 = M([&] { return scale(3.f, sqr(a.w)); });
        Sym f2 = M([&] { return scale(6.f, a.w); });
        return junary(a, f, f1, f2);
    }
    SJet jsqr(const SJet& a) {
        Sym f = M([&] { return sqr(a.w); });
        Sym f1 = M([&] { return scale(2.f, a.w); });
        return junary(a, f, f1, C(2.f));
    }
};

// ------------------------------------------------------------------------------------------ model SLPs
// (restated from the paper, shared with nothing)
using JV = std::vector<SJet>;

// quad12 vector field, state order of PAPER.md:L538: xi = (p[3], phi, theta, psi, v[3], p, q, r), nu = (T, tau[3]);
// eq. (38a) L534 is garbled, the standard ZYX rigid-body form is used (reading R6).  coup: spring force per axis or NULL.
void quad12_field(Builder& B, const Model& M, const SJet* xi, const SJet* nu, const SJet* coup, SJet* out) {
    SJet sphi, cphi, sth, cth, spsi, cpsi;
    B.jsincos(xi[3], &sphi, &cphi);
    B.jsincos(xi[4], &sth, &cth);
    B.jsincos(xi[5], &spsi, &cpsi);
    SJet rcth = B.jrecip(cth);
    const SJet &p = xi[9], &q = xi[10], &r = xi[11];
    SJet a = B.jadd(B.jmul(q, sphi), B.jmul(r, cphi));
    out[0] = xi[6];
    out[1] = xi[7];
    out[2] = xi[8];
    out[3] = B.jadd(p, B.jmul(a, B.jmul(sth, rcth)));
    out[4] = B.jsub(B.jmul(q, cphi), B.jmul(r, sphi));
    out[5] = B.jmul(a, rcth);
    SJet Tm = B.jscale(M.inv_m, nu[0]);
    out[6] = B.jmul(Tm, B.jadd(B.jmul(B.jmul(cpsi, sth), cphi), B.jmul(spsi, sphi)));
    out[7] = B.jmul(Tm, B.jsub(B.jmul(B.jmul(spsi, sth), cphi), B.jmul(cpsi, sphi)));
    out[8] = B.jaddc(B.jmul(Tm, B.jmul(cth, cphi)), -M.g);
    out[9] = B.jadd(B.jscale(M.cp, B.jmul(q, r)), B.jscale(M.iJx, nu[1]));
    out[10] = B.jadd(B.jscale(M.cq, B.jmul(p, r)), B.jscale(M.iJy, nu[2]));
    out[11] = B.jadd(B.jscale(M.cr, B.jmul(p, q)), B.jscale(M.iJz, nu[3]));
    if (coup)
        for (int c = 0; c < 3; ++c) out[6 + c] = B.jadd(out[6 + c], B.jscale(M.inv_m, coup[c]));
}

// chain vector field (BASELINE config 4): spring i joins units i and i+1 per axis, s = k1 d + k3 d^3, d = p_{i+1} - p_i;
// force +s on unit i, -s on unit i+1 (open chain, zero rest length)
void chain_field(Builder& B, const Model& M, const JV& x, const JV& u, JV& out) {
    const int U = M.n_units;
    JV s(3 * std::max(U - 1, 1));
    for (int i = 0; i + 1 < U; ++i)
        for (int c = 0; c < 3; ++c) {
            SJet d = B.jsub(x[12 * (i + 1) + c], x[12 * i + c]);
            s[3 * i + c] = B.jadd(B.jscale(M.k1, d), B.jscale(M.k3, B.jcube(d)));
        }
    for (int i = 0; i < U; ++i) {
        SJet coup[3];
        bool any = false;
        for (int c = 0; c < 3; ++c) {
            if (i + 1 < U && i > 0) { coup[c] = B.jsub(s[3 * i + c], s[3 * (i - 1) + c]); any = true; }
            else if (i + 1 < U) { coup[c] = s[3 * i + c]; any = true; }
            else if (i > 0) { coup[c] = B.jneg(s[3 * (i - 1) + c]); any = true; }
        }
        quad12_field(B, M, &x[12 * i], &u[4 * i], any ? coup : nullptr, &out[12 * i]);
    }
}

// coupled 3-D quadrotors (39)-(42) PAPER.md:L540-558: centroid spring-damper a_i = -alpha U (p_i - pbar) - gamma (v_i - vbar)
// added to the acceleration of unit i; k1 = alpha, k3 = gamma
void centroid_field(Builder& B, const Model& M, const JV& x, const JV& u, JV& out) {
    const int U = M.n_units;
    SJet pbar[3], vbar[3];
    for (int c = 0; c < 3; ++c) {
        SJet sp = x[c], sv = x[6 + c];
        for (int i = 1; i < U; ++i) { sp = B.jadd(sp, x[12 * i + c]); sv = B.jadd(sv, x[12 * i + 6 + c]); }
        pbar[c] = B.jscale(1.f / (float)U, sp);
        vbar[c] = B.jscale(1.f / (float)U, sv);
    }
    for (int i = 0; i < U; ++i) {
        quad12_field(B, M, &x[12 * i], &u[4 * i], nullptr, &out[12 * i]);
        for (int c = 0; c < 3; ++c) {
            SJet a = B.jadd(B.jscale(-M.k1 * (float)U, B.jsub(x[12 * i + c], pbar[c])), B.jscale(-M.k3, B.jsub(x[12 * i + 6 + c], vbar[c])));
            out[12 * i + 6 + c] = B.jadd(out[12 * i + 6 + c], a);
        }
    }
}

// planar quadrotor (37a) PAPER.md:L521-528: x = (px, py, phi, vx, vy, phidot), u = (u1, u2)
void planar_quad_field(Builder& B, const Model& M, const JV& x, const JV& u, JV& out) {
    SJet s, c;
    B.jsincos(x[2], &s, &c);
    SJet thrust = B.jscale(M.inv_m, B.jadd(u[0], u[1]));
    out[0] = x[3];
    out[1] = x[4];
    out[2] = x[5];
    out[3] = B.jneg(B.jmul(thrust, s));
    out[4] = B.jaddc(B.jmul(thrust, c), -M.g);
    out[5] = B.jscale(M.k1, B.jsub(u[1], u[0]));      // k1 holds L / J
}

// satellite (36) PAPER.md:L507-519: x = (q[4], om[3]), u = torque[3];
// qdot = zeta(om) q, omdot = I^-1 (u - om x (I om)), I = diag(Jx, Jy, Jz)
void satellite_field(Builder& B, const Model& M, const JV& x, const JV& u, JV& out) {
    const SJet *q = &x[0], *om = &x[4];
    auto half = [&](const SJet& a) { return B.jscale(0.5f, a); };
    out[0] = half(B.jsub(B.jsub(B.jneg(B.jmul(om[0], q[1])), B.jmul(om[1], q[2])), B.jmul(om[2], q[3])));
    out[1] = half(B.jsub(B.jadd(B.jmul(om[0], q[0]), B.jmul(om[2], q[2])), B.jmul(om[1], q[3])));
    out[2] = half(B.jadd(B.jsub(B.jmul(om[1], q[0]), B.jmul(om[2], q[1])), B.jmul(om[0], q[3])));
    out[3] = half(B.jsub(B.jadd(B.jmul(om[2], q[0]), B.jmul(om[1], q[1])), B.jmul(om[0], q[2])));
    // om x (I om) = ((Jz - Jy) om2 om3, (Jx - Jz) om3 om1, (Jy - Jx) om1 om2); cp, cq, cr hold -(that)/J*
    out[4] = B.jadd(B.jscale(M.cp, B.jmul(om[1], om[2])), B.jscale(M.iJx, u[0]));
    out[5] = B.jadd(B.jscale(M.cq, B.jmul(om[0], om[2])), B.jscale(M.iJy, u[1]));
    out[6] = B.jadd(B.jscale(M.cr, B.jmul(om[0], om[1])), B.jscale(M.iJz, u[2]));
}

void vector_field(Builder& B, const Model& M, const JV& x, const JV& u, JV& out) {
    if (M.id == LEB_MODEL_PLANAR_QUAD) planar_quad_field(B, M, x, u, out);
    else if (M.id == LEB_MODEL_SATELLITE) satellite_field(B, M, x, u, out);
    else if (M.id == LEB_MODEL_QUADCENTROID) centroid_field(B, M, x, u, out);
    else chain_field(B, M, x, u, out);
}

// discrete-time map f(a), a = [x; u]; Euler (the paper's choice, L505) or classical RK4 with u held
void model_f(Builder& B, const Model& M, JV& f) {
    const int n = M.n, N = M.N;
    JV al(N);
    for (int g = 0; g < N; ++g) al[g] = B.in(g);
    if (M.id == LEB_MODEL_UNICYCLE) {
        // a = (px, py, th, v, om); f = (px + dt v cos th, py + dt v sin th, th + dt om)
        SJet s, c;
        B.jsincos(al[2], &s, &c);
        f[0] = B.jadd(al[0], B.jscale(M.dt, B.jmul(al[3], c)));
        f[1] = B.jadd(al[1], B.jscale(M.dt, B.jmul(al[3], s)));
        f[2] = B.jadd(al[2], B.jscale(M.dt, al[4]));
        return;
    }
    JV x(al.begin(), al.begin() + n), u(al.begin() + n, al.end());
    JV k1(n), k2(n), k3(n), k4(n), xs(n);
    vector_field(B, M, x, u, k1);
    if (M.integ == LEB_INTEG_EULER) {
        for (int i = 0; i < n; ++i) f[i] = B.jadd(x[i], B.jscale(M.dt, k1[i]));
        return;
    }
    for (int i = 0; i < n; ++i) xs[i] = B.jadd(x[i], B.jscale(M.half_dt, k1[i]));
    vector_field(B, M, xs, u, k2);
    for (int i = 0; i < n; ++i) xs[i] = B.jadd(x[i], B.jscale(M.half_dt, k2[i]));
    vector_field(B, M, xs, u, k3);
    for (int i = 0; i < n; ++i) xs[i] = B.jadd(x[i], B.jscale(M.dt, k3[i]));
    vector_field(B, M, xs, u, k4);
    for (int i = 0; i < n; ++i)
        f[i] = B.jadd(x[i], B.jscale(M.dt6, B.jadd(B.jadd(B.jadd(k1[i], B.jscale(2.f, k2[i])), B.jscale(2.f, k3[i])), k4[i])));
}

// ------------------------------------------------------------------------------------------ layout
struct RawSeg { std::vector<Ins> ins; std::vector<uint32_t> b; };      // ins: w0 = op, w1 = a (tagged)

inline bool op_has_a(uint32_t op) { return op >= OP_ADD && op != OP_COUNT; }      // a is a slot
inline bool op_has_b(uint32_t op) { return op == OP_ADD || op == OP_SUB || op == OP_MUL || op == OP_MULACC; }   // b is a slot

// Peephole: [q; p = a * b (or c * a); s = q + p] with p used by s only and q, p, s consecutive  ->  [q; s = MULACC / SCALEACC].
// ins: w0 = op, w1 = a; operands that are results of this list carry `tag` (tag | index).  ext[i] != 0: result i is also
// read from outside the list (a WJ slot read by a K segment).  Both interval operations are executed unchanged inside the
// fused instruction, so the enclosure is bit-identical; what goes is one dispatch, one slot and one ring round trip.
void fuse_mul_add(std::vector<Ins>& ins, std::vector<uint32_t>& b, uint32_t tag, const std::vector<uint8_t>* ext,
                  std::vector<uint32_t>* remap_out) {
    const size_t nI = ins.size();
    auto local = [&](uint32_t s) { return tag ? (s & tag) != 0 : true; };
    auto idx = [&](uint32_t s) { return tag ? (s & ~tag) : s; };
    std::vector<uint32_t> uses(nI, 0);
    for (size_t i = 0; i < nI; ++i) {
        const uint32_t op = ins[i].w0;
        if (op_has_a(op) && local(ins[i].w1)) ++uses[idx(ins[i].w1)];
        if (op_has_b(op) && local(b[i])) ++uses[idx(b[i])];
    }
    std::vector<Ins> o;
    std::vector<uint32_t> ob, map(nI, 0), src;          // src: old index of each kept instruction
    o.reserve(nI); ob.reserve(nI); src.reserve(nI);
    auto ref = [&](uint32_t s) { return local(s) ? (tag | map[idx(s)]) : s; };
    for (size_t i = 0; i < nI; ++i) {
        const uint32_t op = ins[i].w0;
        uint32_t a = ins[i].w1, bb = b[i];
        if (op_has_a(op)) a = ref(a);
        if (op_has_b(op)) bb = ref(bb);
        if (op == OP_ADD && o.size() >= 2 && local(a) && local(bb)) {
            const uint32_t last = (uint32_t)o.size() - 1;
            uint32_t ia = idx(a), ib = idx(bb);
            if (ib == last - 1 && ia == last) std::swap(ia, ib);             // interval addition is symmetric
            const uint32_t pop = o[last].w0, qop = o[last - 1].w0;
            const bool p_private = uses[src[last]] == 1 && !(ext && (*ext)[src[last]]);
            if (ia == last - 1 && ib == last && (pop == OP_MUL || pop == OP_SCALE) && qop != OP_OUT && p_private) {
                o[last].w0 = pop == OP_MUL ? OP_MULACC : OP_SCALEACC;
                map[i] = last;
                // the fused instruction now stands for s: it inherits s's uses
                src[last] = (uint32_t)i;
                continue;
            }
        }
        map[i] = (uint32_t)o.size();
        o.push_back(Ins{op, a});
        ob.push_back(bb);
        src.push_back((uint32_t)i);
    }
    ins.swap(o);
    b.swap(ob);
    if (remap_out) remap_out->swap(map);
}

}  // namespace

// Compile the model into a tape.  with_mu: non-centred boxes (25a) L272 (reading R4: prefix hull sets).
void leb_compile_tape(const Model& M, bool with_mu, Tape* T) {
    const int n = M.n, N = M.N;
    *T = Tape();
    T->n = n; T->N = N; T->uses_mu = with_mu;
    auto& task_out = T->task_out;
    auto& task_var = T->task_var;

    // ---- first-order dependencies: which outputs read coordinate g at all (pass WJ in direction g)
    std::vector<std::vector<uint8_t>> dep(N, std::vector<uint8_t>(n, 0));
    {
        for (int g = 0; g < N; ++g) {
            Builder B;
            B.j = g; B.k = -1; B.use_mu = with_mu;
            B.in_slot.assign(N, -1);
            JV f(n);
            model_f(B, M, f);
            for (int l = 0; l < n; ++l) dep[g][l] = f[l].wj.k != SK_Z;
        }
    }


    for (int j = 0; j < N; ++j) {
        Builder B;
        B.j = j; B.k = -1; B.use_mu = with_mu;
        B.in_slot.assign(N, -1);
        JV f(n);
        model_f(B, M, f);                       // pass WJ: memo filled
        Sym Dj = S(B.emit(with_mu ? OP_DELTAMU : OP_DELTA, (uint32_t)j, 0));

        std::vector<RawSeg> ksegs;
        std::vector<uint8_t> wj_live(B.wj_ins.size() + 64, 0), wj_kuse(B.wj_ins.size() + 64, 0);
        std::vector<int> acc_of(n, -1);
        int n_acc = 0;
        for (int k = j; k < N; ++k) {
            bool share = false;
            for (int l = 0; l < n && !share; ++l) share = dep[j][l] && dep[k][l];
            if (!share) continue;
            B.kphase = true; B.diag = (k == j); B.k = k; B.mpos = 0;
            B.k_ins.clear(); B.k_b.clear(); B.const_k.clear();
            JV fk(n);
            model_f(B, M, fk);
            // terms of eq. (15): off-diagonal [H_kj] D_j D_k, diagonal 1/2 [H_kk] sqr(D_k)   (D_k^2 >= 0, L152)
            Sym fac;
            bool have_fac = false;
            for (int l = 0; l < n; ++l) {
                if (fk[l].wjk.k == SK_Z) continue;
                if (!have_fac) {
                    if (B.diag) fac = B.sqr(Dj);
                    else fac = B.mul(Dj, S(B.emit(with_mu ? OP_DELTAMU : OP_DELTA, (uint32_t)k, 0)));
                    have_fac = true;
                }
                Sym t = B.mul(fk[l].wjk, fac);
                if (B.diag) t = B.scale(0.5f, t);
                t = B.mat(t);
                if (acc_of[l] < 0) acc_of[l] = n_acc++;
                B.emit(OP_OUT, t.s, ((uint32_t)l << 16) | (uint32_t)acc_of[l]);
            }
            B.kphase = false;
            if (!have_fac) continue;
            // ---- dead code: keep what the OUT instructions read
            const size_t nk = B.k_ins.size();
            std::vector<uint8_t> live(nk, 0);
            auto touch = [&](uint32_t s) { if (s & KTAG) live[s & ~KTAG] = 1; else { wj_live[s] = 1; wj_kuse[s] = 1; } };
            for (size_t i = nk; i-- > 0;) {
                const uint32_t op = B.k_ins[i].w0;
                if (op == OP_OUT) live[i] = 1;
                if (!live[i]) continue;
                if (op_has_a(op)) touch(B.k_ins[i].w1);
                if (op_has_b(op)) touch(B.k_b[i]);
            }
            RawSeg seg;
            std::vector<uint32_t> remap(nk, 0);
            for (size_t i = 0; i < nk; ++i) {
                if (!live[i]) continue;
                remap[i] = (uint32_t)seg.ins.size();
                seg.ins.push_back(B.k_ins[i]);
                seg.b.push_back(B.k_b[i]);
            }
            for (size_t i = 0; i < seg.ins.size(); ++i) {
                const uint32_t op = seg.ins[i].w0;
                if (op_has_a(op) && (seg.ins[i].w1 & KTAG)) seg.ins[i].w1 = KTAG | remap[seg.ins[i].w1 & ~KTAG];
                if (op_has_b(op) && (seg.b[i] & KTAG)) seg.b[i] = KTAG | remap[seg.b[i] & ~KTAG];
            }
            fuse_mul_add(seg.ins, seg.b, KTAG, nullptr, nullptr);
            ksegs.push_back(std::move(seg));
        }
        if (ksegs.empty()) continue;
        // ---- dead code in WJ
        const size_t nw = B.wj_ins.size();
        wj_live.resize(nw, 0);
        for (size_t i = nw; i-- > 0;) {
            if (!wj_live[i]) continue;
            const uint32_t op = B.wj_ins[i].w0;
            if (op_has_a(op)) wj_live[B.wj_ins[i].w1] = 1;
            if (op_has_b(op)) wj_live[B.wj_b[i]] = 1;
        }
        // compact the live WJ instructions, fuse, and keep the composed renumbering for the K segments
        std::vector<uint32_t> wremap(nw, 0);
        Task task{};
        task.j = (uint32_t)j;
        task.wj_begin = (uint32_t)T->ins.size();
        uint32_t nwj = 0;
        for (size_t i = 0; i < nw; ++i) if (wj_live[i]) wremap[i] = nwj++;
        std::vector<Ins> wins;
        std::vector<uint32_t> wb;
        std::vector<uint8_t> wext;
        wins.reserve(nwj); wb.reserve(nwj); wext.reserve(nwj);
        for (size_t i = 0; i < nw; ++i) {
            if (!wj_live[i]) continue;
            const uint32_t op = B.wj_ins[i].w0;
            uint32_t a = B.wj_ins[i].w1, b = B.wj_b[i];
            if (op_has_a(op)) a = wremap[a];
            if (op_has_b(op)) b = wremap[b];
            wins.push_back(Ins{op, a});
            wb.push_back(b);
            wext.push_back(wj_kuse[i]);
        }
        {
            std::vector<uint32_t> remap2;
            fuse_mul_add(wins, wb, 0u, &wext, &remap2);
            for (size_t i = 0; i < nw; ++i) if (wj_live[i]) wremap[i] = remap2[wremap[i]];
            nwj = (uint32_t)wins.size();
        }
        task.wj_count = nwj;
        // gradient rows: one per input coordinate this task reads
        std::vector<int> grow(N, -1);
        int n_grad = 0;
        auto grad_row = [&](uint32_t g) { if (grow[g] < 0) grow[g] = n_grad++; return (uint32_t)grow[g]; };
        auto is_input = [](uint32_t op) { return op == OP_BOX || op == OP_PT || op == OP_DELTA || op == OP_BOXMU || op == OP_DELTAMU; };
        uint64_t cost = 0;
        double flops = 0.0;
        for (size_t i = 0; i < wins.size(); ++i) {
            const uint32_t op = wins[i].w0;
            uint32_t a = wins[i].w1, b = wb[i];
            if (is_input(op)) b = grad_row(a);
            T->ins.push_back(Ins{op | (a << 8), b});
            ++cost; flops += op_flops(op);
        }
        task.seg_begin = (uint32_t)T->segs.size();
        uint32_t max_k = 0;
        for (auto& seg : ksegs) {
            Seg sg{(uint32_t)T->ins.size(), (uint32_t)seg.ins.size()};
            max_k = std::max(max_k, sg.count);
            auto fix = [&](uint32_t s) { return (s & KTAG) ? nwj + (s & ~KTAG) : wremap[s]; };
            for (size_t i = 0; i < seg.ins.size(); ++i) {
                const uint32_t op = seg.ins[i].w0;
                uint32_t a = seg.ins[i].w1, b = seg.b[i];
                if (op_has_a(op)) a = fix(a);
                if (op_has_b(op)) b = fix(b);
                if (is_input(op)) b = grad_row(a);
                T->ins.push_back(Ins{op | (a << 8), b});
                ++cost; flops += op_flops(op);
            }
            T->segs.push_back(sg);
        }
        task.seg_count = (uint32_t)ksegs.size();
        // ---- operand sources and FAR bits (an_tape.h)
        {
            Ins* base = T->ins.data();
            auto src_of = [&](uint32_t slot, uint32_t user, uint32_t seg_dst0, uint32_t seg_begin) -> uint32_t {
                if (slot < seg_dst0) { base[task.wj_begin + slot].w0 |= OP_FAR; return SRC_GLOBAL; }     // WJ slot read by a K segment
                if (user - slot == 1 && (base[seg_begin + (slot - seg_dst0)].w0 & OP_MASK) != OP_OUT) return SRC_PREV;
                if (user - slot < kRing) return SRC_RING;
                base[seg_begin + (slot - seg_dst0)].w0 |= OP_FAR;
                return SRC_GLOBAL;
            };
            auto scan = [&](uint32_t begin, uint32_t count, uint32_t dst0) {
                for (uint32_t i = 0; i < count; ++i) {
                    const uint32_t op = base[begin + i].w0 & OP_MASK;
                    if (op_has_a(op)) base[begin + i].w0 |= src_of(base[begin + i].w0 >> 8, dst0 + i, dst0, begin) << SRC_SHIFT;
                    if (op_has_b(op)) base[begin + i].w1 |= src_of(base[begin + i].w1 & B_MASK, dst0 + i, dst0, begin) << B_SRC_SHIFT;
                }
            };
            scan(task.wj_begin, nwj, 0);
            for (uint32_t q = 0; q < task.seg_count; ++q) scan(T->segs[task.seg_begin + q].begin, T->segs[task.seg_begin + q].count, nwj);
        }
        task.n_slots = nwj + max_k;
        task.acc_base = 0; task.n_acc = (uint32_t)n_acc;          // row bases are assigned per task set (leb_build_taskset)
        task.grad_base = 0; task.n_grad = (uint32_t)n_grad;
        task.cost = (uint32_t)std::min<uint64_t>(cost, 0xffffffffu);
        {   // which output / input each of this task's rows belongs to (for the reduction tables)
            std::vector<uint32_t> to(n_acc), tv(n_grad);
            for (int l = 0; l < n; ++l) if (acc_of[l] >= 0) to[acc_of[l]] = (uint32_t)l;
            for (int g = 0; g < N; ++g) if (grow[g] >= 0) tv[grow[g]] = (uint32_t)g;
            task_out.push_back(std::move(to));
            task_var.push_back(std::move(tv));
        }
        T->flops_fwd += flops;
        T->max_slots = std::max(T->max_slots, task.n_slots);
        T->max_acc = std::max(T->max_acc, task.n_acc);
        T->max_grad = std::max(T->max_grad, task.n_grad);
        T->base.push_back(task);
        T->ins_fwd += cost;
    }
}

void leb_build_taskset(const Tape& T, uint32_t target, TaskSet* set) {
    const int n = T.n, N = T.N;
    *set = TaskSet();
    std::vector<uint32_t> parent;
    for (size_t q = 0; q < T.base.size(); ++q) {
        const Task& tk = T.base[q];
        if (tk.cost <= target) { set->tasks.push_back(tk); parent.push_back((uint32_t)q); continue; }
        // parts of about equal K cost, each at most `target` (but never shorter than the WJ they repeat)
        const uint32_t kcost = tk.cost - tk.wj_count;
        const uint32_t room = std::max<uint32_t>(target > tk.wj_count ? target - tk.wj_count : 0, tk.wj_count);
        const uint32_t parts = (kcost + room - 1) / room;
        const uint32_t per = (kcost + parts - 1) / parts;
        uint32_t s0 = 0;
        while (s0 < tk.seg_count) {
            uint32_t s1 = s0, c = 0, mk = 0;
            while (s1 < tk.seg_count && (s1 == s0 || c + T.segs[tk.seg_begin + s1].count <= per)) {
                c += T.segs[tk.seg_begin + s1].count;
                mk = std::max(mk, T.segs[tk.seg_begin + s1].count);
                ++s1;
            }
            Task part = tk;
            part.seg_begin = tk.seg_begin + s0;
            part.seg_count = s1 - s0;
            part.n_slots = tk.wj_count + mk;
            part.cost = tk.wj_count + c;
            set->tasks.push_back(part);
            parent.push_back((uint32_t)q);
            s0 = s1;
        }
    }
    // rows are handed out in creation order (ascending j), so every reduction adds in ascending j
    std::vector<std::vector<uint32_t>> orow(n), vrow(N);
    uint32_t ar = 0, gr = 0;
    for (size_t q = 0; q < set->tasks.size(); ++q) {
        Task& tk = set->tasks[q];
        tk.acc_base = ar; tk.grad_base = gr;
        const auto& to = T.task_out[parent[q]];
        const auto& tv = T.task_var[parent[q]];
        for (uint32_t r = 0; r < tk.n_acc; ++r) orow[to[r]].push_back(ar + r);
        for (uint32_t r = 0; r < tk.n_grad; ++r) vrow[tv[r]].push_back(gr + r);
        ar += tk.n_acc; gr += tk.n_grad;
        set->ins_fwd += tk.cost;
    }
    set->acc_rows = ar; set->grad_rows = gr;
    set->out_ptr.assign(n + 1, 0);
    for (int l = 0; l < n; ++l) { set->out_ptr[l] = (uint32_t)set->out_rows.size(); set->out_rows.insert(set->out_rows.end(), orow[l].begin(), orow[l].end()); }
    set->out_ptr[n] = (uint32_t)set->out_rows.size();
    set->var_ptr.assign(N + 1, 0);
    for (int g = 0; g < N; ++g) { set->var_ptr[g] = (uint32_t)set->var_rows.size(); set->var_rows.insert(set->var_rows.end(), vrow[g].begin(), vrow[g].end()); }
    set->var_ptr[N] = (uint32_t)set->var_rows.size();
    // heavy tasks first (the device pulls tasks from a counter)
    std::stable_sort(set->tasks.begin(), set->tasks.end(), [](const Task& a, const Task& b) { return a.cost > b.cost; });
}

}  // namespace leb_an

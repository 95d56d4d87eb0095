// analytic.cu -- leb_analytic_fwd / leb_vjp(kind 0): path-based interval-Hessian bound (Thm 1, eq. (15),
// PAPER.md:L164-167) and its VJP, as an interpreter of the interval tape of an_tape.h / an_compile.cu.
//
// Work decomposition: a TASK is one path index j of the tape (its segment WJ(j) and its segments K(j,k));
// a warp takes a (task, group of 32 tiles) work item from a counter, heavy tasks first.  Lane = tile: the tape is
// the same for every tile, so a warp executes one instruction stream on 32 sets of intervals -- no divergence
// except on data-dependent selections inside an instruction.  Slots live in a per-warp region of a global
// workspace laid out [slot][lane] (256-byte coalesced accesses, L1/L2 resident while hot).  FP32 with directed
// rounding throughout: lower endpoints round down, upper endpoints round up, sinf / cosf are padded by their
// 2-ulp error bound, so every enclosure contains the exact-arithmetic enclosure of the same tape (steps A1-A3 of
// SURVEY 8(a)).  A task leaves its partial sums of eq. (15) in a buffer; a second kernel adds the partial rows of
// every output in ascending j with RD / RU (a fixed order: results are bitwise reproducible).
//
// VJP: the same forward sweep keeps every slot (SSA), then the tape is walked backwards with one adjoint per slot
// endpoint; min / max / hull selections are re-derived from the stored primal values (ties -> the first candidate
// in the order lo*lo, lo*hi, hi*lo, hi*hi; reading R20).  The K segments are run forward and backward one
// at a time, their adjoints flowing into WJ(j)'s, which is reversed once at the end of the task.  Per-task input
// adjoints go to a partial-gradient buffer and are summed in a fixed order as well.
#include <new>
#include "an_tape.h"
#include "internal.h"

namespace leb_an {

constexpr int kWarpsPerBlock = 4;
constexpr unsigned FULL = 0xffffffffu;

struct DevTape {
    const uint2* ins;
    const Seg* segs;
    const Task* tasks;
    const uint32_t *out_ptr, *out_rows, *var_ptr, *var_rows;
    int ntasks, n, N;
};

struct VmArgs {
    int tiles, ngroups, tiles_pad;
    const float *nom, *rad, *mu;
    int ld_in;
    const float *g_lo, *g_hi;
    int ld_out;
    float2* partial;        // forward: [acc_rows][tiles_pad] (lo, hi); VJP: [grad_rows][tiles_pad] (nom_bar, rad_bar)
    float* partial_mu;      // VJP with mu: [grad_rows][tiles_pad]
    float2* ws;             // per-warp slot regions
    size_t ws_stride;       // float2 elements per warp region
    uint32_t adj_off, acc_off, gm_off;   // slot offsets inside a region: adjoint file; accumulator rows (forward) or
                                         // (nom_bar, rad_bar) rows (VJP); (mu_bar, -) rows (VJP)
    unsigned* counter;
    int* tile_bad;
};

// ------------------------------------------------------------------ interval primitives (directed rounding)
__device__ __forceinline__ float pad_dn(float s) { return fmaxf(-1.f, __fadd_rd(s, -(fabsf(s) * 3.0e-7f + 1e-30f))); }
__device__ __forceinline__ float pad_up(float s) { return fminf(1.f, __fadd_ru(s, (fabsf(s) * 3.0e-7f + 1e-30f))); }
// does [lo, hi] contain a point c + 2 pi k ?  (FP64 test with a tiny outward slack: when in doubt say yes,
// which only widens the enclosure by O(slack^2))
__device__ __forceinline__ bool contains_2pik(float lo, float hi, double c) {
    const double INV_TWO_PI = 0.15915494309189533576888376337251;
    double a = ((double)lo - c) * INV_TWO_PI - 1e-9, b = ((double)hi - c) * INV_TWO_PI + 1e-9;
    return floor(b) >= ceil(a);
}
__device__ __forceinline__ float2 iv_mul(float2 a, float2 b) {
    float lo = fminf(fminf(__fmul_rd(a.x, b.x), __fmul_rd(a.x, b.y)), fminf(__fmul_rd(a.y, b.x), __fmul_rd(a.y, b.y)));
    float hi = fmaxf(fmaxf(__fmul_ru(a.x, b.x), __fmul_ru(a.x, b.y)), fmaxf(__fmul_ru(a.y, b.x), __fmul_ru(a.y, b.y)));
    return make_float2(lo, hi);
}
__device__ __forceinline__ float2 iv_sqr(float2 a) {
    if (a.x >= 0.f) return make_float2(__fmul_rd(a.x, a.x), __fmul_ru(a.y, a.y));
    if (a.y <= 0.f) return make_float2(__fmul_rd(a.y, a.y), __fmul_ru(a.x, a.x));
    return make_float2(0.f, fmaxf(__fmul_ru(a.x, a.x), __fmul_ru(a.y, a.y)));
}
// x^3 is increasing; for x < 0 the lower bound is -(up(|x|^3))
__device__ __forceinline__ float cube_dn(float x) {
    if (x >= 0.f) return __fmul_rd(__fmul_rd(x, x), x);
    float m = -x;
    return -__fmul_ru(__fmul_ru(m, m), m);
}
__device__ __forceinline__ float cube_up(float x) {
    if (x >= 0.f) return __fmul_ru(__fmul_ru(x, x), x);
    float m = -x;
    return -__fmul_rd(__fmul_rd(m, m), m);
}
constexpr double HALF_PI = 1.5707963267948966192313216916398;
constexpr double PI_D = 3.1415926535897932384626433832795;

__device__ __forceinline__ float2 iv_sin(float2 a) {
    const bool has_max = contains_2pik(a.x, a.y, HALF_PI), has_min = contains_2pik(a.x, a.y, -HALF_PI);
    const float sl = sinf(a.x), sh = sinf(a.y);
    return make_float2(has_min ? -1.f : fminf(pad_dn(sl), pad_dn(sh)), has_max ? 1.f : fmaxf(pad_up(sl), pad_up(sh)));
}
__device__ __forceinline__ float2 iv_cos(float2 a) {
    const bool has_max = contains_2pik(a.x, a.y, 0.0), has_min = contains_2pik(a.x, a.y, PI_D);
    const float cl = cosf(a.x), ch = cosf(a.y);
    return make_float2(has_min ? -1.f : fminf(pad_dn(cl), pad_dn(ch)), has_max ? 1.f : fmaxf(pad_up(cl), pad_up(ch)));
}

__device__ __forceinline__ float as_f(uint32_t u) { return __uint_as_float(u); }

// ------------------------------------------------------------------ forward sweep of one segment
// S: global slot file of this lane (slot s at S[s * 32]); rb: shared-memory address of this lane's column of the warp's
// ring (slot s at rb + (s % kRing) * 256); dst0: slot of the segment's first instruction.  Where an operand comes from
// (the previous result, the ring, the global file) was decided by the compiler (an_tape.h).  VJP: every primal value
// is also kept in the global file (the reverse sweep needs it), the adjoint of a FAR slot is cleared, OUT does nothing.
__device__ __forceinline__ void prefetch_row(const float2* row) {
    asm volatile("prefetch.global.L1 [%0];" ::"l"(row));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(row + 16));
}
__device__ __forceinline__ float2 lds2(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts2(uint32_t addr, float2 v) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y));
}
__device__ __forceinline__ float2 fetch(uint32_t src, uint32_t slot, const float2& prev, uint32_t rb, const float2* __restrict__ S) {
    if (src == SRC_PREV) return prev;
    if (src == SRC_RING) return lds2(rb + (slot & (kRing - 1)) * 256u);
    return S[(size_t)slot * 32];
}

template <bool VJP>
__device__ __forceinline__ void run_fwd(const uint2* __restrict__ ins, uint32_t begin, uint32_t count, uint32_t dst0,
                                        float2* __restrict__ S, uint32_t rb, const VmArgs& A,
                                        const float* __restrict__ nom, const float* __restrict__ rad,
                                        const float* __restrict__ mu, bool& bad, int lane) {
    float2* ADJ = S + (size_t)A.adj_off * 32;
    float2* ACC = S + (size_t)A.acc_off * 32;
    const float2* row0 = S - lane;
    float2 prev = make_float2(0.f, 0.f);
    uint32_t dst = dst0;
    uint2 nxt = make_uint2(0u, 0u);
    if ((uint32_t)lane < count) nxt = __ldg(ins + begin + lane);
    for (uint32_t base = 0; base < count; base += 32) {
        const uint2 mine = nxt;
        nxt = make_uint2(0u, 0u);
        if (base + 32 + lane < count) {
            // next chunk: fetch its instructions and pull its global operands towards L1 while this chunk executes
            nxt = __ldg(ins + begin + base + 32 + lane);
            const uint32_t op = nxt.x & OP_MASK;
            if (op >= OP_ADD && ((nxt.x >> SRC_SHIFT) & 3u) == SRC_GLOBAL) prefetch_row(row0 + (size_t)(nxt.x >> 8) * 32);
            if ((op == OP_ADD || op == OP_SUB || op == OP_MUL || op == OP_MULACC) && (nxt.y >> B_SRC_SHIFT) == SRC_GLOBAL) prefetch_row(row0 + (size_t)(nxt.y & B_MASK) * 32);
        }
        const int m = min(32u, count - base);
        for (int i = 0; i < m; ++i, ++dst) {
            const uint32_t w0 = __shfl_sync(FULL, mine.x, i), w1 = __shfl_sync(FULL, mine.y, i);
            const uint32_t op = w0 & OP_MASK, a = w0 >> 8;
            float2 r;
            if (op == OP_MUL) {
                const float2 x = fetch((w0 >> SRC_SHIFT) & 3u, a, prev, rb, S), y = fetch(w1 >> B_SRC_SHIFT, w1 & B_MASK, prev, rb, S);
                r = iv_mul(x, y);
            } else if (op == OP_MULACC) {
                const float2 x = fetch((w0 >> SRC_SHIFT) & 3u, a, prev, rb, S), y = fetch(w1 >> B_SRC_SHIFT, w1 & B_MASK, prev, rb, S);
                const float2 p = iv_mul(x, y);
                r = make_float2(__fadd_rd(prev.x, p.x), __fadd_ru(prev.y, p.y));
            } else if (op == OP_SCALE || op == OP_SCALEACC) {
                const float2 x = fetch((w0 >> SRC_SHIFT) & 3u, a, prev, rb, S);
                const float c = as_f(w1);
                r = c >= 0.f ? make_float2(__fmul_rd(c, x.x), __fmul_ru(c, x.y)) : make_float2(__fmul_rd(c, x.y), __fmul_ru(c, x.x));
                if (op == OP_SCALEACC) r = make_float2(__fadd_rd(prev.x, r.x), __fadd_ru(prev.y, r.y));
            } else if (op == OP_ADD) {
                const float2 x = fetch((w0 >> SRC_SHIFT) & 3u, a, prev, rb, S), y = fetch(w1 >> B_SRC_SHIFT, w1 & B_MASK, prev, rb, S);
                r = make_float2(__fadd_rd(x.x, y.x), __fadd_ru(x.y, y.y));
            } else if (op == OP_OUT) {
                const float2 x = fetch((w0 >> SRC_SHIFT) & 3u, a, prev, rb, S);
                if (!VJP) {
                    float2* p = ACC + (size_t)(w1 & 0xffffu) * 32;
                    const float2 c = *p;
                    *p = make_float2(__fadd_rd(c.x, x.x), __fadd_ru(c.y, x.y));
                }
                prev = x;
                continue;
            } else {
                float2 x = make_float2(0.f, 0.f);
                if (op >= OP_ADD) x = fetch((w0 >> SRC_SHIFT) & 3u, a, prev, rb, S);
                switch (op) {
                    case OP_BOX: { float c = nom[a], s = rad[a]; r = make_float2(__fadd_rd(c, -s), __fadd_ru(c, s)); break; }
                    case OP_PT: { float c = nom[a]; r = make_float2(c, c); break; }
                    case OP_DELTA: { float s = rad[a]; r = make_float2(-s, s); break; }
                    case OP_BOXMU: {   // hull of [c + mu - s, c + mu + s] and {c}: the segment from a~ to a point of the box
                        float c = nom[a], s = rad[a], u = mu[a];
                        r = make_float2(__fadd_rd(c, fminf(__fadd_rd(u, -s), 0.f)), __fadd_ru(c, fmaxf(__fadd_ru(u, s), 0.f)));
                        break;
                    }
                    case OP_DELTAMU: { float s = rad[a], u = mu[a]; r = make_float2(__fadd_rd(u, -s), __fadd_ru(u, s)); break; }
                    case OP_CONST: { float c = as_f(w1); r = make_float2(c, c); break; }
                    case OP_SUB: {
                        const float2 y = fetch(w1 >> B_SRC_SHIFT, w1 & B_MASK, prev, rb, S);
                        r = make_float2(__fadd_rd(x.x, -y.y), __fadd_ru(x.y, -y.x));
                        break;
                    }
                    case OP_NEG: r = make_float2(-x.y, -x.x); break;
                    case OP_ADDC: { float c = as_f(w1); r = make_float2(__fadd_rd(x.x, c), __fadd_ru(x.y, c)); break; }
                    case OP_SQR: r = iv_sqr(x); break;
                    case OP_CUBE: r = make_float2(cube_dn(x.x), cube_up(x.y)); break;
                    case OP_RECIP:
                        if (x.x <= 0.f && x.y >= 0.f) { bad = true; r = make_float2(1.f, 1.f); }
                        else r = make_float2(__frcp_rd(x.y), __frcp_ru(x.x));
                        break;
                    case OP_SIN: r = iv_sin(x); break;
                    case OP_COS: r = iv_cos(x); break;
                    default: r = make_float2(0.f, 0.f); break;
                }
            }
            sts2(rb + (dst & (kRing - 1)) * 256u, r);
            if (VJP || (w0 & OP_FAR)) S[(size_t)dst * 32] = r;
            if (VJP && (w0 & OP_FAR)) ADJ[(size_t)dst * 32] = make_float2(0.f, 0.f);
            prev = r;
        }
    }
}

// ------------------------------------------------------------------ reverse sweep of one segment
// The adjoint of a slot is the sum of what its uses send back.  Uses fewer than kRing instructions later (same segment:
// operand sources PREV / RING) accumulate in the shared-memory ring; every other use adds into the global adjoint file
// with a fire-and-forget reduction (each lane owns its column: no contention), and only FAR slots read it back.
__device__ __forceinline__ void red_add(float2* p, float dl, float dh) { atomicAdd(p, make_float2(dl, dh)); }
__device__ __forceinline__ void send(uint32_t src, uint32_t slot, float dl, float dh, uint32_t rb, float2* __restrict__ ADJ) {
    if (src != SRC_GLOBAL) {
        const uint32_t p = rb + (slot & (kRing - 1)) * 256u;
        float2 v = lds2(p);
        v.x += dl; v.y += dh;
        sts2(p, v);
    } else {
        red_add(ADJ + (size_t)slot * 32, dl, dh);
    }
}

__device__ __forceinline__ void run_bwd(const uint2* __restrict__ ins, uint32_t begin, uint32_t count, uint32_t dst0,
                                        float2* __restrict__ S, uint32_t rb, const VmArgs& A,
                                        const float* __restrict__ rad, const float* __restrict__ mu,
                                        const float* __restrict__ g_lo, const float* __restrict__ g_hi, int lane) {
    float2* ADJ = S + (size_t)A.adj_off * 32;
    float2* G0 = S + (size_t)A.acc_off * 32;                 // (nom_bar, rad_bar) per gradient row
    float2* GM = S + (size_t)A.gm_off * 32;                  // (mu_bar, -) per gradient row
    const float2* row0 = S - lane;
    if (count == 0) return;
    for (uint32_t q = 0; q < kRing; ++q) sts2(rb + q * 256u, make_float2(0.f, 0.f));
    const int last = (int)((count - 1) / 32) * 32;
    uint2 nxt = make_uint2(0u, 0u);
    if ((uint32_t)last + lane < count) nxt = __ldg(ins + begin + last + lane);
    for (int base = last; base >= 0; base -= 32) {
        const uint2 mine = nxt;
        // this chunk's primal operands towards L1 (they were written by the forward sweep, long ago)
        if ((uint32_t)base + lane < count) {
            const uint32_t op = mine.x & OP_MASK;
            if (op == OP_MUL || op == OP_MULACC || op == OP_SQR || op == OP_CUBE || op == OP_SIN || op == OP_COS) prefetch_row(row0 + (size_t)(mine.x >> 8) * 32);
            if (op == OP_MUL || op == OP_MULACC) prefetch_row(row0 + (size_t)(mine.y & B_MASK) * 32);
            if (op == OP_RECIP) prefetch_row(row0 + (size_t)(dst0 + base + lane) * 32);
        }
        nxt = make_uint2(0u, 0u);
        if (base >= 32) nxt = __ldg(ins + begin + base - 32 + lane);
        const int m = min(32u, count - (uint32_t)base);
        for (int i = m - 1; i >= 0; --i) {
            const uint32_t w0 = __shfl_sync(FULL, mine.x, i), w1 = __shfl_sync(FULL, mine.y, i);
            const uint32_t op = w0 & OP_MASK, a = w0 >> 8, sa = (w0 >> SRC_SHIFT) & 3u;
            const uint32_t dst = dst0 + (uint32_t)base + (uint32_t)i;
            const uint32_t rp = rb + (dst & (kRing - 1)) * 256u;
            if (op == OP_OUT) {
                const uint32_t l = w1 >> 16;
                send(sa, a, g_lo[l], g_hi[l], rb, ADJ);
                continue;                                    // an OUT slot has no uses: its ring entry is still zero
            }
            float2 d = lds2(rp);
            sts2(rp, make_float2(0.f, 0.f));                 // the ring entry now belongs to slot dst - kRing
            if (w0 & OP_FAR) { const float2 g = __ldcg(ADJ + (size_t)dst * 32); d.x += g.x; d.y += g.y; }
            const float dl = d.x, dh = d.y;
            if (dl == 0.f && dh == 0.f) continue;
            if (op == OP_MUL || op == OP_MULACC) {
                if (op == OP_MULACC) send(SRC_RING, dst - 1, dl, dh, rb, ADJ);       // the running sum passes the adjoint on
                const uint32_t b = w1 & B_MASK, sb = w1 >> B_SRC_SHIFT;
                const float2 x = S[(size_t)a * 32], y = S[(size_t)b * 32];
                // lower endpoint: first minimum of (xl yl, xl yh, xh yl, xh yh), products rounded down as in the forward
                float best = __fmul_rd(x.x, y.x); int sl = 0;
                float p = __fmul_rd(x.x, y.y); if (p < best) { best = p; sl = 1; }
                p = __fmul_rd(x.y, y.x); if (p < best) { best = p; sl = 2; }
                p = __fmul_rd(x.y, y.y); if (p < best) { best = p; sl = 3; }
                best = __fmul_ru(x.x, y.x); int sh = 0;
                p = __fmul_ru(x.x, y.y); if (p > best) { best = p; sh = 1; }
                p = __fmul_ru(x.y, y.x); if (p > best) { best = p; sh = 2; }
                p = __fmul_ru(x.y, y.y); if (p > best) { best = p; sh = 3; }
                const float xs_l = (sl & 2) ? x.y : x.x, ys_l = (sl & 1) ? y.y : y.x;
                const float xs_h = (sh & 2) ? x.y : x.x, ys_h = (sh & 1) ? y.y : y.x;
                float2 ax = make_float2(0.f, 0.f), ay = make_float2(0.f, 0.f);
                if (sl & 2) ax.y += dl * ys_l; else ax.x += dl * ys_l;
                if (sl & 1) ay.y += dl * xs_l; else ay.x += dl * xs_l;
                if (sh & 2) ax.y += dh * ys_h; else ax.x += dh * ys_h;
                if (sh & 1) ay.y += dh * xs_h; else ay.x += dh * xs_h;
                send(sa, a, ax.x, ax.y, rb, ADJ);
                send(sb, b, ay.x, ay.y, rb, ADJ);
                continue;
            }
            if (op == OP_SCALE || op == OP_SCALEACC) {
                if (op == OP_SCALEACC) send(SRC_RING, dst - 1, dl, dh, rb, ADJ);
                const float c = as_f(w1);
                if (c >= 0.f) send(sa, a, c * dl, c * dh, rb, ADJ);
                else send(sa, a, c * dh, c * dl, rb, ADJ);
                continue;
            }
            if (op == OP_ADD) {
                send(sa, a, dl, dh, rb, ADJ);
                send(w1 >> B_SRC_SHIFT, w1 & B_MASK, dl, dh, rb, ADJ);
                continue;
            }
            switch (op) {
                case OP_BOX: red_add(G0 + (size_t)w1 * 32, dl + dh, dh - dl); break;
                case OP_PT: red_add(G0 + (size_t)w1 * 32, dl + dh, 0.f); break;
                case OP_DELTA: red_add(G0 + (size_t)w1 * 32, 0.f, dh - dl); break;
                case OP_BOXMU: {
                    // lo = c + min(mu - s, 0), hi = c + max(mu + s, 0); ties keep the first candidate
                    const float s = rad[a], u = mu[a];
                    const float fl = (0.f < __fadd_rd(u, -s)) ? 0.f : dl, fh = (0.f > __fadd_ru(u, s)) ? 0.f : dh;
                    red_add(G0 + (size_t)w1 * 32, dl + dh, fh - fl);
                    red_add(GM + (size_t)w1 * 32, fl + fh, 0.f);
                    break;
                }
                case OP_DELTAMU:
                    red_add(G0 + (size_t)w1 * 32, 0.f, dh - dl);
                    red_add(GM + (size_t)w1 * 32, dl + dh, 0.f);
                    break;
                case OP_SUB: send(sa, a, dl, dh, rb, ADJ); send(w1 >> B_SRC_SHIFT, w1 & B_MASK, -dh, -dl, rb, ADJ); break;
                case OP_NEG: send(sa, a, -dh, -dl, rb, ADJ); break;
                case OP_ADDC: send(sa, a, dl, dh, rb, ADJ); break;
                case OP_SQR: {
                    const float2 x = S[(size_t)a * 32];
                    if (x.x >= 0.f) send(sa, a, 2.f * x.x * dl, 2.f * x.y * dh, rb, ADJ);
                    else if (x.y <= 0.f) send(sa, a, 2.f * x.x * dh, 2.f * x.y * dl, rb, ADJ);
                    else if (__fmul_ru(x.y, x.y) > __fmul_ru(x.x, x.x)) send(sa, a, 0.f, 2.f * x.y * dh, rb, ADJ);
                    else send(sa, a, 2.f * x.x * dh, 0.f, rb, ADJ);
                    break;
                }
                case OP_CUBE: {
                    const float2 x = S[(size_t)a * 32];
                    send(sa, a, 3.f * x.x * x.x * dl, 3.f * x.y * x.y * dh, rb, ADJ);
                    break;
                }
                case OP_RECIP: {
                    const float2 r = S[(size_t)dst * 32];          // (1/hi, 1/lo)
                    send(sa, a, -dh * r.y * r.y, -dl * r.x * r.x, rb, ADJ);
                    break;
                }
                case OP_SIN: {
                    const float2 x = S[(size_t)a * 32];
                    const bool has_max = contains_2pik(x.x, x.y, HALF_PI), has_min = contains_2pik(x.x, x.y, -HALF_PI);
                    const float sl = sinf(x.x), sh = sinf(x.y);
                    float al = 0.f, ah = 0.f;
                    if (!has_min) { if (pad_dn(sh) < pad_dn(sl)) ah += cosf(x.y) * dl; else al += cosf(x.x) * dl; }
                    if (!has_max) { if (pad_up(sh) > pad_up(sl)) ah += cosf(x.y) * dh; else al += cosf(x.x) * dh; }
                    send(sa, a, al, ah, rb, ADJ);
                    break;
                }
                case OP_COS: {
                    const float2 x = S[(size_t)a * 32];
                    const bool has_max = contains_2pik(x.x, x.y, 0.0), has_min = contains_2pik(x.x, x.y, PI_D);
                    const float cl = cosf(x.x), ch = cosf(x.y);
                    float al = 0.f, ah = 0.f;
                    if (!has_min) { if (pad_dn(ch) < pad_dn(cl)) ah -= sinf(x.y) * dl; else al -= sinf(x.x) * dl; }
                    if (!has_max) { if (pad_up(ch) > pad_up(cl)) ah -= sinf(x.y) * dh; else al -= sinf(x.x) * dh; }
                    send(sa, a, al, ah, rb, ADJ);
                    break;
                }
                default: break;
            }
        }
    }
}

// ------------------------------------------------------------------ the interpreter kernel
template <bool VJP>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 3) an_vm_kernel(DevTape P, VmArgs A) {
    extern __shared__ float2 ring[];                         // [kWarpsPerBlock][kRing][32]
    const int lane = threadIdx.x & 31;
    const size_t wid = (size_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
    float2* S = A.ws + wid * A.ws_stride + lane;
    const uint32_t R = (uint32_t)__cvta_generic_to_shared(ring + (size_t)(threadIdx.x >> 5) * kRing * 32 + lane);
    const unsigned nwork = (unsigned)P.ntasks * (unsigned)A.ngroups;
    for (;;) {
        unsigned t = 0;
        if (lane == 0) t = atomicAdd(A.counter, 1u);
        t = __shfl_sync(FULL, t, 0);
        if (t >= nwork) break;
        const Task tk = P.tasks[t / A.ngroups];
        const int tile = (int)(t % A.ngroups) * 32 + lane;
        const bool valid = tile < A.tiles;
        const size_t row = (size_t)(valid ? tile : A.tiles - 1);
        const float* nom = A.nom + row * A.ld_in;
        const float* rad = A.rad + row * A.ld_in;
        const float* mu = A.mu ? A.mu + row * A.ld_in : nullptr;
        bool bad = false;
        if (!VJP) {
            float2* ACC = S + (size_t)A.acc_off * 32;
            for (uint32_t r = 0; r < tk.n_acc; ++r) ACC[(size_t)r * 32] = make_float2(0.f, 0.f);
            run_fwd<false>(P.ins, tk.wj_begin, tk.wj_count, 0, S, R, A, nom, rad, mu, bad, lane);
            for (uint32_t q = 0; q < tk.seg_count; ++q) {
                const Seg sg = P.segs[tk.seg_begin + q];
                run_fwd<false>(P.ins, sg.begin, sg.count, tk.wj_count, S, R, A, nom, rad, mu, bad, lane);
            }
            if (valid)
                for (uint32_t r = 0; r < tk.n_acc; ++r) A.partial[(size_t)(tk.acc_base + r) * A.tiles_pad + tile] = ACC[(size_t)r * 32];
        } else {
            float2* G0 = S + (size_t)A.acc_off * 32;
            float2* GM = S + (size_t)A.gm_off * 32;
            const float* g_lo = A.g_lo + row * A.ld_out;
            const float* g_hi = A.g_hi + row * A.ld_out;
            for (uint32_t r = 0; r < tk.n_grad; ++r) { G0[(size_t)r * 32] = make_float2(0.f, 0.f); GM[(size_t)r * 32] = make_float2(0.f, 0.f); }
            run_fwd<true>(P.ins, tk.wj_begin, tk.wj_count, 0, S, R, A, nom, rad, mu, bad, lane);
            for (uint32_t q = 0; q < tk.seg_count; ++q) {
                const Seg sg = P.segs[tk.seg_begin + q];
                run_fwd<true>(P.ins, sg.begin, sg.count, tk.wj_count, S, R, A, nom, rad, mu, bad, lane);
                run_bwd(P.ins, sg.begin, sg.count, tk.wj_count, S, R, A, rad, mu, g_lo, g_hi, lane);
            }
            run_bwd(P.ins, tk.wj_begin, tk.wj_count, 0, S, R, A, rad, mu, g_lo, g_hi, lane);
            if (valid)
                for (uint32_t r = 0; r < tk.n_grad; ++r) {
                    A.partial[(size_t)(tk.grad_base + r) * A.tiles_pad + tile] = __ldcg(G0 + (size_t)r * 32);
                    if (A.partial_mu) A.partial_mu[(size_t)(tk.grad_base + r) * A.tiles_pad + tile] = __ldcg(GM + (size_t)r * 32).x;
                }
        }
        if (bad && valid) A.tile_bad[tile] = 1;
    }
}

// ------------------------------------------------------------------ refinements built on forward + VJP (Table II)
// input-domain partitioning: sub-box p of tile t along coordinate g: part q_g = (p / stride_g) % splits_g of splits_g equal
// parts.  The sub-radius is rounded up and padded by a few ulps of the box so that the FP32 sub-boxes cover the box.
__global__ void subbox_kernel(size_t tiles, int P, int N, int ld_in, const int* __restrict__ splits, const int* __restrict__ strides,
                              const float* __restrict__ nom, const float* __restrict__ rad, const float* __restrict__ mu,
                              float* __restrict__ nom_x, float* __restrict__ rad_x, float* __restrict__ mu_x) {
    const size_t total = tiles * (size_t)P * N;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int g = (int)(idx % N);
        const size_t tp = idx / N;
        const int p = (int)(tp % P);
        const size_t t = tp / P;
        const int s = splits[g], q = (p / strides[g]) % s;
        const float r = rad[t * ld_in + g], m = mu ? mu[t * ld_in + g] : 0.f;
        nom_x[idx] = nom[t * ld_in + g];
        if (s == 1) { rad_x[idx] = r; mu_x[idx] = m; continue; }
        const float inv = 1.f / (float)s;
        rad_x[idx] = __fadd_ru(__fmul_ru(r, inv), 4.f * 1.1920929e-07f * (fabsf(m) + r));
        mu_x[idx] = fmaf(r, fmaf((float)(2 * q + 1), inv, -1.f), m);
    }
}

// hull over the P sub-boxes of a tile
__global__ void hull_kernel(size_t tiles, int P, int n, int ld_out, const float* __restrict__ lo_x, const float* __restrict__ hi_x,
                            float* __restrict__ r_lo, float* __restrict__ r_hi) {
    const size_t total = tiles * (size_t)n;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const size_t t = idx / n;
        const int l = (int)(idx - t * n);
        float lo = INFINITY, hi = -INFINITY;
        for (int p = 0; p < P; ++p) {
            const size_t o = (t * P + p) * (size_t)n + l;
            lo = fminf(lo, lo_x[o]);
            hi = fmaxf(hi, hi_x[o]);
            if (!(lo_x[o] == lo_x[o])) { lo = -INFINITY; hi = INFINITY; }
        }
        r_lo[t * ld_out + l] = lo;
        r_hi[t * ld_out + l] = hi;
    }
}

// PGD: mu = centre - nom
// VJP of the hull: the cotangent of r_lo[l] goes to the sub-box with the first minimum, that of r_hi[l] to the first maximum
__global__ void hull_select_kernel(size_t tiles, int P, int n, int ld_out, const float* __restrict__ lo_x, const float* __restrict__ hi_x,
                                   const float* __restrict__ g_lo, const float* __restrict__ g_hi, float* __restrict__ glo_x,
                                   float* __restrict__ ghi_x) {
    const size_t total = tiles * (size_t)n;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const size_t t = idx / n;
        const int l = (int)(idx - t * n);
        float lo = INFINITY, hi = -INFINITY;
        int pl = 0, ph = 0;
        for (int p = 0; p < P; ++p) {
            const size_t o = (t * P + p) * (size_t)n + l;
            if (lo_x[o] < lo) { lo = lo_x[o]; pl = p; }
            if (hi_x[o] > hi) { hi = hi_x[o]; ph = p; }
        }
        const float gl = g_lo[t * ld_out + l], gh = g_hi[t * ld_out + l];
        for (int p = 0; p < P; ++p) {
            const size_t o = (t * P + p) * (size_t)n + l;
            glo_x[o] = p == pl ? gl : 0.f;
            ghi_x[o] = p == ph ? gh : 0.f;
        }
    }
}
// chain the sub-box gradients back through subbox_kernel's formulas, sub-boxes added in ascending order (reproducible)
__global__ void subbox_vjp_kernel(size_t tiles, int P, int N, int ld_in, const int* __restrict__ splits, const int* __restrict__ strides,
                                  const float* __restrict__ mu, const float* __restrict__ gn_x, const float* __restrict__ gr_x,
                                  const float* __restrict__ gm_x, float* __restrict__ grad_nom, float* __restrict__ grad_rad,
                                  float* __restrict__ grad_mu) {
    const size_t total = tiles * (size_t)N;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const size_t t = idx / N;
        const int g = (int)(idx - t * N);
        const int s = splits[g], stride = strides[g];
        const float inv = 1.f / (float)s, eps4 = 4.f * 1.1920929e-07f;
        const float m = mu ? mu[t * ld_in + g] : 0.f, sg = (m > 0.f) - (m < 0.f);
        float an = 0.f, ar = 0.f, am = 0.f;
        for (int p = 0; p < P; ++p) {
            const size_t o = (t * P + p) * (size_t)N + g;
            const float gn = gn_x[o], gr = gr_x[o], gm = gm_x[o];
            an += gn;
            if (s == 1) { ar += gr; am += gm; continue; }
            const int q = (p / stride) % s;
            ar += gr * (inv + eps4) + gm * fmaf((float)(2 * q + 1), inv, -1.f);
            am += gm + gr * eps4 * sg;
        }
        grad_nom[t * ld_in + g] = an;
        grad_rad[t * ld_in + g] = ar;
        if (grad_mu) grad_mu[t * ld_in + g] = am;
    }
}

__global__ void pgd_mu_kernel(size_t count, const float* __restrict__ centre, const float* __restrict__ nom, float* __restrict__ mu) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (size_t)gridDim.x * blockDim.x) mu[i] = centre[i] - nom[i];
}
__global__ void fill_kernel(size_t count, float v, float* __restrict__ a) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (size_t)gridDim.x * blockDim.x) a[i] = v;
}
// one block per tile: width of the enclosure, keep the best iterate, take the projected gradient step
__global__ void pgd_step_kernel(int n, int N, int ld_in, int first, int last, float lr, const float* __restrict__ lo,
                                const float* __restrict__ hi, const float* __restrict__ gn, const float* __restrict__ gm,
                                const float* __restrict__ centre, const float* __restrict__ eps, float* __restrict__ cur,
                                float* __restrict__ best_nom, float* __restrict__ w0, float* __restrict__ wbest) {
    __shared__ float red[32];
    __shared__ int take;
    const size_t t = blockIdx.x;
    float w = 0.f;
    for (int l = threadIdx.x; l < n; l += blockDim.x) w += hi[t * n + l] - lo[t * n + l];
    for (int off = 16; off; off >>= 1) w += __shfl_xor_sync(FULL, w, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = w;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) tot += red[q];
        if (first) { w0[t] = tot; wbest[t] = tot; take = 1; }
        else if (tot < wbest[t]) { wbest[t] = tot; take = 1; }
        else take = 0;
    }
    __syncthreads();
    for (int g = threadIdx.x; g < N; g += blockDim.x) {
        const size_t o = t * ld_in + g;
        const float x = cur[o];
        if (take) best_nom[o] = x;
        if (!last) {
            const float d = gn[o] - gm[o];            // d W / d a~ with the box fixed (mu = centre - a~)
            float y = x - lr * d;
            y = fminf(fmaxf(y, centre[o] - eps[o]), centre[o] + eps[o]);
            if (y == y) cur[o] = y;
        }
    }
}

// ------------------------------------------------------------------ fixed-order reductions over the tasks
// one block per tile: validates the tile's inputs, then thread l adds the partial rows of output l in ascending j
__global__ void an_reduce_fwd_kernel(DevTape P, int tiles_pad, const float* __restrict__ nom, const float* __restrict__ rad,
                                     const float* __restrict__ mu, int ld_in, const float2* __restrict__ partial,
                                     const int* __restrict__ tile_bad, float* __restrict__ r_lo, float* __restrict__ r_hi,
                                     int ld_out, int* __restrict__ domain_flag) {
    const int tile = blockIdx.x;
    int bad = 0;
    for (int g = threadIdx.x; g < P.N; g += blockDim.x) {
        const float a = nom[(size_t)tile * ld_in + g], s = rad[(size_t)tile * ld_in + g];
        if (!(fabsf(a) <= 3.0e38f) || !(s >= 0.f) || !(s <= 3.0e38f)) bad = 1;
        if (mu) { const float u = mu[(size_t)tile * ld_in + g]; if (!(fabsf(u) <= 3.0e38f)) bad = 1; }
    }
    bad = __syncthreads_or(bad | (threadIdx.x == 0 ? tile_bad[tile] : 0));
    for (int l = threadIdx.x; l < P.n; l += blockDim.x) {
        float lo = 0.f, hi = 0.f;
        for (uint32_t q = P.out_ptr[l]; q < P.out_ptr[l + 1]; ++q) {
            const float2 v = partial[(size_t)P.out_rows[q] * tiles_pad + tile];
            lo = __fadd_rd(lo, v.x);
            hi = __fadd_ru(hi, v.y);
        }
        if (bad) { lo = -INFINITY; hi = INFINITY; }
        r_lo[(size_t)tile * ld_out + l] = lo;
        r_hi[(size_t)tile * ld_out + l] = hi;
    }
    if (bad && threadIdx.x == 0) atomicExch(domain_flag, 1);
}

__global__ void an_reduce_vjp_kernel(DevTape P, int tiles_pad, const float* __restrict__ nom, const float* __restrict__ rad,
                                     const float* __restrict__ mu, int ld_in, const float2* __restrict__ partial,
                                     const float* __restrict__ partial_mu, const int* __restrict__ tile_bad,
                                     float* __restrict__ grad_nom, float* __restrict__ grad_rad, float* __restrict__ grad_mu,
                                     int* __restrict__ domain_flag) {
    const int tile = blockIdx.x;
    int bad = 0;
    for (int g = threadIdx.x; g < P.N; g += blockDim.x) {
        const float a = nom[(size_t)tile * ld_in + g], s = rad[(size_t)tile * ld_in + g];
        if (!(fabsf(a) <= 3.0e38f) || !(s >= 0.f) || !(s <= 3.0e38f)) bad = 1;
        if (mu) { const float u = mu[(size_t)tile * ld_in + g]; if (!(fabsf(u) <= 3.0e38f)) bad = 1; }
    }
    bad = __syncthreads_or(bad | (threadIdx.x == 0 ? tile_bad[tile] : 0));
    for (int g = threadIdx.x; g < P.N; g += blockDim.x) {
        float gn = 0.f, gr = 0.f, gm = 0.f;
        for (uint32_t q = P.var_ptr[g]; q < P.var_ptr[g + 1]; ++q) {
            const size_t o = (size_t)P.var_rows[q] * tiles_pad + tile;
            const float2 v = partial[o];
            gn += v.x;
            gr += v.y;
            if (partial_mu) gm += partial_mu[o];
        }
        if (bad) { gn = NAN; gr = NAN; gm = NAN; }
        grad_nom[(size_t)tile * ld_in + g] = gn;
        grad_rad[(size_t)tile * ld_in + g] = gr;
        if (grad_mu) grad_mu[(size_t)tile * ld_in + g] = gm;
    }
    if (bad && threadIdx.x == 0) atomicExch(domain_flag, 1);
}

}  // namespace leb_an

// ============================================================================================== host side
using namespace leb_an;

struct DevSet {                   // a TaskSet on the device
    uint32_t target = 0;
    DevTape dev{};
    uint32_t acc_rows = 0, grad_rows = 0, ntasks = 0;
    std::vector<void*> allocs;
};

struct AnState {
    bool ready = false;
    Model model{};
    Tape tape[2];                 // [0] centred boxes, [1] non-centred (mu != NULL), compiled on first use
    bool have[2] = {false, false};
    const uint2* d_ins[2] = {nullptr, nullptr};
    const Seg* d_segs[2] = {nullptr, nullptr};
    std::vector<void*> tape_allocs[2];
    std::vector<DevSet> sets[2];  // task sets built so far (one per cost target, see leb_build_taskset)
    // buffers grown on demand
    float2* ws = nullptr; size_t ws_bytes = 0;
    float2* partial = nullptr; size_t partial_bytes = 0;
    float* partial_mu = nullptr; size_t partial_mu_bytes = 0;
    int* tile_bad = nullptr; size_t tile_bad_n = 0;
    unsigned* counter = nullptr;
    int num_sms = 148;
    bool attr_done = false;
    // scratch of the refinements (partitioning, PGD): grown on demand
    float* scratch[12] = {nullptr};
    size_t scratch_bytes[12] = {0};
    int* d_splits = nullptr;      // [2][N]: splits, strides
    size_t d_splits_n = 0;
};

AnState* leb_an_create() {
    AnState* S = new (std::nothrow) AnState();
    if (!S) return nullptr;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&S->num_sms, cudaDevAttrMultiProcessorCount, dev);
    return S;
}

static void free_tape(AnState* S, int v) {
    for (void* p : S->tape_allocs[v]) cudaFree(p);
    S->tape_allocs[v].clear();
    for (DevSet& d : S->sets[v]) for (void* p : d.allocs) cudaFree(p);
    S->sets[v].clear();
    S->have[v] = false;
}

void leb_an_destroy(AnState* S) {
    if (!S) return;
    free_tape(S, 0); free_tape(S, 1);
    if (S->ws) cudaFree(S->ws);
    if (S->partial) cudaFree(S->partial);
    if (S->partial_mu) cudaFree(S->partial_mu);
    if (S->tile_bad) cudaFree(S->tile_bad);
    if (S->counter) cudaFree(S->counter);
    for (int i = 0; i < 12; ++i) if (S->scratch[i]) cudaFree(S->scratch[i]);
    if (S->d_splits) cudaFree(S->d_splits);
    delete S;
}

bool leb_an_ready(const AnState* S) { return S && S->ready; }
int leb_an_n(const AnState* S) { return S->model.n; }
int leb_an_N(const AnState* S) { return S->model.N; }

template <class T>
static bool upload(std::vector<void*>& allocs, const std::vector<T>& h, const T** d) {
    void* p = nullptr;
    const size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(T);
    if (cudaMalloc(&p, bytes) != cudaSuccess) return false;
    allocs.push_back(p);
    if (!h.empty() && cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return false;
    *d = (const T*)p;
    return true;
}

static leb_status ensure_tape(AnState* S, int v) {
    if (S->have[v]) return LEB_OK;
    Tape& T = S->tape[v];
    leb_compile_tape(S->model, v == 1, &T);
    static_assert(sizeof(Ins) == sizeof(uint2), "Ins is two words");
    std::vector<uint2> raw(T.ins.size());
    for (size_t i = 0; i < T.ins.size(); ++i) raw[i] = make_uint2(T.ins[i].w0, T.ins[i].w1);
    if (!upload(S->tape_allocs[v], raw, &S->d_ins[v]) || !upload(S->tape_allocs[v], T.segs, &S->d_segs[v])) { free_tape(S, v); return LEB_ERR_NOMEM; }
    S->have[v] = true;
    return LEB_OK;
}

// the task set whose longest task has about `target` instructions (targets are rounded down to (4 + m) 2^e, m < 4, at least
// 256 -- a quarter of an octave -- so that only a handful of sets ever exist and the cut does not jump by a factor of two)
static const DevSet* ensure_set(AnState* S, int v, uint64_t target64) {
    uint32_t target = 256;
    while ((uint64_t)target * 2 <= target64 && target < 0x40000000u) target <<= 1;
    for (uint32_t m = 3; m >= 1; --m)
        if ((uint64_t)target + (uint64_t)m * (target / 4) <= target64) { target += m * (target / 4); break; }
    for (const DevSet& d : S->sets[v]) if (d.target == target) return &d;
    const Tape& T = S->tape[v];
    TaskSet set;
    leb_build_taskset(T, target, &set);
    S->sets[v].emplace_back();
    DevSet& D = S->sets[v].back();
    D.target = target;
    D.acc_rows = set.acc_rows; D.grad_rows = set.grad_rows; D.ntasks = (uint32_t)set.tasks.size();
    D.dev.ins = S->d_ins[v]; D.dev.segs = S->d_segs[v];
    D.dev.ntasks = (int)set.tasks.size(); D.dev.n = T.n; D.dev.N = T.N;
    const bool ok = upload(D.allocs, set.tasks, &D.dev.tasks) && upload(D.allocs, set.out_ptr, &D.dev.out_ptr) &&
                    upload(D.allocs, set.out_rows, &D.dev.out_rows) && upload(D.allocs, set.var_ptr, &D.dev.var_ptr) &&
                    upload(D.allocs, set.var_rows, &D.dev.var_rows);
    if (!ok) { for (void* p : D.allocs) cudaFree(p); S->sets[v].pop_back(); return nullptr; }
    return &D;
}

leb_status leb_an_set_model(AnState* S, const Model& M) {
    free_tape(S, 0); free_tape(S, 1);
    S->model = M;
    S->ready = true;
    if (!S->counter && cudaMalloc(&S->counter, sizeof(unsigned)) != cudaSuccess) return LEB_ERR_NOMEM;
    return ensure_tape(S, 0);
}

template <class T>
static bool grow(T** p, size_t* have, size_t need_bytes) {
    if (*have >= need_bytes) return true;
    if (*p) { cudaDeviceSynchronize(); cudaFree(*p); *p = nullptr; *have = 0; }
    if (cudaMalloc((void**)p, need_bytes) != cudaSuccess) return false;
    *have = need_bytes;
    return true;
}

void leb_an_stats(const AnState* S, double* flops_fwd, long long* ins_fwd, long long* tape_ins, int* ntasks, int* max_slots) {
    const Tape& T = S->tape[0];
    *flops_fwd = T.flops_fwd; *ins_fwd = (long long)T.ins_fwd; *tape_ins = (long long)T.ins.size();
    *ntasks = (int)T.base.size(); *max_slots = (int)T.max_slots;
}

// forward (g_lo == NULL) or VJP
static leb_status an_run(AnState* S, bool vjp, int tiles, const float* nom, const float* rad, const float* mu, int ld_in,
                         float* r_lo, float* r_hi, const float* g_lo, const float* g_hi, int ld_out, float* grad_nom,
                         float* grad_rad, float* grad_mu, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof) {
    if (tiles == 0) return LEB_OK;
    const int v = mu ? 1 : 0;
    leb_status es = ensure_tape(S, v);
    if (es != LEB_OK) return es;
    const Tape& T = S->tape[v];
    VmArgs A{};
    A.tiles = tiles; A.ngroups = (tiles + 31) / 32; A.tiles_pad = A.ngroups * 32;
    A.nom = nom; A.rad = rad; A.mu = mu; A.ld_in = ld_in; A.g_lo = g_lo; A.g_hi = g_hi; A.ld_out = ld_out;
    // work items = (task, group of 32 tiles).  A small batch cannot fill the GPU with whole tasks -- its run time would be
    // the longest task's -- so tasks longer than the per-warp share of the work are cut (leb_build_taskset)
    const int warps_resident = S->num_sms * 3 * kWarpsPerBlock;
    const DevSet* DS = ensure_set(S, v, T.ins_fwd * (uint64_t)A.ngroups / (uint64_t)warps_resident);
    if (!DS) return LEB_ERR_NOMEM;
    const DevTape& D = DS->dev;
    const size_t nwork = (size_t)DS->ntasks * A.ngroups;
    // slot regions
    size_t region;     // float2 elements per lane
    if (!vjp) { A.adj_off = 0; A.acc_off = T.max_slots; A.gm_off = 0; region = (size_t)T.max_slots + T.max_acc; }
    else { A.adj_off = T.max_slots; A.acc_off = 2 * T.max_slots; A.gm_off = 2 * T.max_slots + T.max_grad; region = 2 * (size_t)T.max_slots + 2 * (size_t)T.max_grad; }
    region = std::max<size_t>(region, 1);
    A.ws_stride = region * 32;
    int blocks = S->num_sms * 3;      // 64 KB of ring per block: three blocks (12 warps) per SM
    const size_t need_blocks = (nwork + kWarpsPerBlock - 1) / kWarpsPerBlock;
    if ((size_t)blocks > need_blocks) blocks = (int)std::max<size_t>(need_blocks, 1);
    const size_t rows = vjp ? DS->grad_rows : DS->acc_rows;
    if (!grow(&S->ws, &S->ws_bytes, (size_t)blocks * kWarpsPerBlock * A.ws_stride * sizeof(float2))) return LEB_ERR_NOMEM;
    if (!grow(&S->partial, &S->partial_bytes, std::max<size_t>(rows, 1) * A.tiles_pad * sizeof(float2))) return LEB_ERR_NOMEM;
    if (vjp && mu && !grow(&S->partial_mu, &S->partial_mu_bytes, std::max<size_t>(rows, 1) * A.tiles_pad * sizeof(float))) return LEB_ERR_NOMEM;
    {
        size_t have = S->tile_bad_n * sizeof(int);
        if (!grow(&S->tile_bad, &have, (size_t)A.tiles_pad * sizeof(int))) return LEB_ERR_NOMEM;
        S->tile_bad_n = have / sizeof(int);
    }
    A.ws = S->ws; A.partial = S->partial; A.partial_mu = (vjp && mu) ? S->partial_mu : nullptr;
    A.counter = S->counter; A.tile_bad = S->tile_bad;
    cudaMemsetAsync(S->counter, 0, sizeof(unsigned), st);
    cudaMemsetAsync(S->tile_bad, 0, (size_t)A.tiles_pad * sizeof(int), st);
    const int kc = vjp ? LEB_KC_ANALYTIC_VJP : LEB_KC_ANALYTIC_FWD;
    prof->begin(kc, st);
    if (nwork > 0) {
        const size_t smem = (size_t)kWarpsPerBlock * kRing * 32 * sizeof(float2);
        if (!S->attr_done) {      // per context, hence per device
            if (cudaFuncSetAttribute(an_vm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
                cudaFuncSetAttribute(an_vm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
                return LEB_ERR_CUDA;
            S->attr_done = true;
        }
        if (vjp) an_vm_kernel<true><<<blocks, kWarpsPerBlock * 32, smem, st>>>(D, A);
        else an_vm_kernel<false><<<blocks, kWarpsPerBlock * 32, smem, st>>>(D, A);
        ++*launches;
    }
    // algorithmic work: the tape's FP32 operations per tile (the reverse sweep is counted as twice the forward)
    prof->end(kc, st, (vjp ? 3.0 : 1.0) * T.flops_fwd * tiles);
    const int threads = 128;
    if (vjp) an_reduce_vjp_kernel<<<tiles, threads, 0, st>>>(D, A.tiles_pad, nom, rad, mu, ld_in, S->partial, A.partial_mu, S->tile_bad, grad_nom, grad_rad, grad_mu, domain_flag);
    else an_reduce_fwd_kernel<<<tiles, threads, 0, st>>>(D, A.tiles_pad, nom, rad, mu, ld_in, S->partial, S->tile_bad, r_lo, r_hi, ld_out, domain_flag);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

static float* scratch(AnState* S, int slot, size_t count) {
    if (!grow(&S->scratch[slot], &S->scratch_bytes[slot], std::max<size_t>(count, 4) * sizeof(float))) return nullptr;
    return S->scratch[slot];
}
static unsigned gs_blocks(size_t work) { return (unsigned)std::min<size_t>((work + 255) / 256, 148 * 16); }

// input-domain partitioning: hull of the bounds of the grid of sub-boxes, every sub-box a non-centred box
// about the same nominal point
// the (splits | strides) table of a partition on the device; *P_out = sub-boxes per tile
static leb_status upload_splits(AnState* S, int tiles, const int* splits_host, long long* P_out, cudaStream_t st) {
    const int N = S->model.N;
    std::vector<int> tab(2 * (size_t)N);
    long long P = 1;
    for (int g = N - 1; g >= 0; --g) {
        if (splits_host[g] < 1) return LEB_ERR_ARG;
        tab[g] = splits_host[g];
        tab[N + g] = (int)P;
        P *= splits_host[g];
        if (P > 65536) return LEB_ERR_SHAPE;
    }
    if ((long long)tiles * P > 2000000000LL) return LEB_ERR_SHAPE;
    if (S->d_splits_n < 2 * (size_t)N) {
        if (S->d_splits) { cudaDeviceSynchronize(); cudaFree(S->d_splits); S->d_splits = nullptr; }
        if (cudaMalloc(&S->d_splits, 2 * (size_t)N * sizeof(int)) != cudaSuccess) return LEB_ERR_NOMEM;
        S->d_splits_n = 2 * (size_t)N;
    }
    cudaStreamSynchronize(st);        // the table of a previous call may still be in use
    if (cudaMemcpy(S->d_splits, tab.data(), 2 * (size_t)N * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) return LEB_ERR_CUDA;
    *P_out = P;
    return LEB_OK;
}

leb_status leb_an_partition(AnState* S, int tiles, const float* nom, const float* rad, const float* mu, int ld_in,
                            const int* splits_host, float* r_lo, float* r_hi, int ld_out, int* domain_flag, cudaStream_t st,
                            long long* launches, LebProf* prof) {
    if (tiles == 0) return LEB_OK;
    const int N = S->model.N, n = S->model.n;
    long long P = 1;
    leb_status us = upload_splits(S, tiles, splits_host, &P, st);
    if (us != LEB_OK) return us;
    const size_t xt = (size_t)tiles * (size_t)P;
    float *nx = scratch(S, 0, xt * N), *rx = scratch(S, 1, xt * N), *mx = scratch(S, 2, xt * N), *lx = scratch(S, 3, xt * n), *hx = scratch(S, 4, xt * n);
    if (!nx || !rx || !mx || !lx || !hx) return LEB_ERR_NOMEM;
    subbox_kernel<<<gs_blocks(xt * N), 256, 0, st>>>((size_t)tiles, (int)P, N, ld_in, S->d_splits, S->d_splits + N, nom, rad, mu, nx, rx, mx);
    ++*launches;
    leb_status es = an_run(S, false, (int)xt, nx, rx, mx, N, lx, hx, nullptr, nullptr, n, nullptr, nullptr, nullptr, domain_flag, st, launches, prof);
    if (es != LEB_OK) return es;
    hull_kernel<<<gs_blocks((size_t)tiles * n), 256, 0, st>>>((size_t)tiles, (int)P, n, ld_out, lx, hx, r_lo, r_hi);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

// VJP of the partitioned bound: sub-boxes forward, the hull's selection, the ordinary VJP on the sub-boxes with the selected
// cotangents, and the chain rule of the sub-box construction
leb_status leb_an_partition_vjp(AnState* S, int tiles, const float* nom, const float* rad, const float* mu, int ld_in,
                                const int* splits_host, const float* g_lo, const float* g_hi, int ld_out, float* grad_nom,
                                float* grad_rad, float* grad_mu, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof) {
    if (tiles == 0) return LEB_OK;
    const int N = S->model.N, n = S->model.n;
    long long P = 1;
    leb_status us = upload_splits(S, tiles, splits_host, &P, st);
    if (us != LEB_OK) return us;
    const size_t xt = (size_t)tiles * (size_t)P;
    float *nx = scratch(S, 0, xt * N), *rx = scratch(S, 1, xt * N), *mx = scratch(S, 2, xt * N), *lx = scratch(S, 3, xt * n), *hx = scratch(S, 4, xt * n);
    float *gnx = scratch(S, 5, xt * N), *grx = scratch(S, 6, xt * N), *glx = scratch(S, 7, xt * n), *ghx = scratch(S, 8, xt * n), *gmx = scratch(S, 9, xt * N);
    if (!nx || !rx || !mx || !lx || !hx || !gnx || !grx || !glx || !ghx || !gmx) return LEB_ERR_NOMEM;
    subbox_kernel<<<gs_blocks(xt * N), 256, 0, st>>>((size_t)tiles, (int)P, N, ld_in, S->d_splits, S->d_splits + N, nom, rad, mu, nx, rx, mx);
    ++*launches;
    leb_status es = an_run(S, false, (int)xt, nx, rx, mx, N, lx, hx, nullptr, nullptr, n, nullptr, nullptr, nullptr, domain_flag, st, launches, prof);
    if (es != LEB_OK) return es;
    hull_select_kernel<<<gs_blocks((size_t)tiles * n), 256, 0, st>>>((size_t)tiles, (int)P, n, ld_out, lx, hx, g_lo, g_hi, glx, ghx);
    ++*launches;
    es = an_run(S, true, (int)xt, nx, rx, mx, N, nullptr, nullptr, glx, ghx, n, gnx, grx, gmx, domain_flag, st, launches, prof);
    if (es != LEB_OK) return es;
    subbox_vjp_kernel<<<gs_blocks((size_t)tiles * N), 256, 0, st>>>((size_t)tiles, (int)P, N, ld_in, S->d_splits, S->d_splits + N, mu, gnx, grx, gmx,
                                                                  grad_nom, grad_rad, grad_mu);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

// nominal refinement by projected gradient descent (Table II): box (centre, rad) fixed, nominal point inside
// |a~ - centre| <= eps, objective = total width of the enclosure of the remainder about a~
leb_status leb_an_pgd(AnState* S, int tiles, const float* centre, const float* rad, const float* eps, int ld_in, int steps, float lr,
                      float* nom, float* w0, float* wbest, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof) {
    if (tiles == 0) return LEB_OK;
    const int N = S->model.N, n = S->model.n;
    const size_t ci = (size_t)tiles * ld_in, co = (size_t)tiles * n;
    float *cur = scratch(S, 0, ci), *mu = scratch(S, 1, ci), *gn = scratch(S, 2, ci), *gr = scratch(S, 5, ci), *gm = scratch(S, 6, ci);
    float *lo = scratch(S, 3, co), *hi = scratch(S, 4, co), *glo = scratch(S, 7, co), *ghi = scratch(S, 8, co);
    if (!cur || !mu || !gn || !gr || !gm || !lo || !hi || !glo || !ghi) return LEB_ERR_NOMEM;
    if (cudaMemcpyAsync(cur, nom, ci * sizeof(float), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return LEB_ERR_CUDA;
    fill_kernel<<<gs_blocks(co), 256, 0, st>>>(co, -1.f, glo);
    fill_kernel<<<gs_blocks(co), 256, 0, st>>>(co, 1.f, ghi);
    cudaMemsetAsync(gn, 0, ci * sizeof(float), st);
    cudaMemsetAsync(gm, 0, ci * sizeof(float), st);
    *launches += 2;
    for (int it = 0; it <= steps; ++it) {
        pgd_mu_kernel<<<gs_blocks(ci), 256, 0, st>>>(ci, centre, cur, mu);
        ++*launches;
        leb_status es = an_run(S, false, tiles, cur, rad, mu, ld_in, lo, hi, nullptr, nullptr, n, nullptr, nullptr, nullptr, domain_flag, st, launches, prof);
        if (es != LEB_OK) return es;
        if (it < steps) {
            es = an_run(S, true, tiles, cur, rad, mu, ld_in, nullptr, nullptr, glo, ghi, n, gn, gr, gm, domain_flag, st, launches, prof);
            if (es != LEB_OK) return es;
        }
        pgd_step_kernel<<<tiles, 128, 0, st>>>(n, N, ld_in, it == 0, it == steps, lr, lo, hi, gn, gm, centre, eps, cur, nom, w0, wbest);
        ++*launches;
    }
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_an_forward(AnState* S, int tiles, const float* nom, const float* rad, const float* mu, int ld_in, float* r_lo,
                          float* r_hi, int ld_out, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof) {
    return an_run(S, false, tiles, nom, rad, mu, ld_in, r_lo, r_hi, nullptr, nullptr, ld_out, nullptr, nullptr, nullptr, domain_flag, st, launches, prof);
}

leb_status leb_an_vjp(AnState* S, int tiles, const float* nom, const float* rad, const float* mu, const float* g_lo, const float* g_hi,
                      int ld_in, int ld_out, float* grad_nom, float* grad_rad, float* grad_mu, int* domain_flag, cudaStream_t st,
                      long long* launches, LebProf* prof) {
    return an_run(S, true, tiles, nom, rad, mu, ld_in, nullptr, nullptr, g_lo, g_hi, ld_out, grad_nom, grad_rad, grad_mu, domain_flag, st, launches, prof);
}

Model leb_make_model(const leb_analytic_model& m) {
    Model M{};
    M.id = m.model_id;
    M.integ = (m.model_id == LEB_MODEL_UNICYCLE) ? LEB_INTEG_EULER : m.integ;
    M.n_units = (m.model_id == LEB_MODEL_QUADCHAIN || m.model_id == LEB_MODEL_QUADCENTROID) ? m.n_units : 1;
    switch (m.model_id) {
        case LEB_MODEL_UNICYCLE: M.n = 3; M.N = 5; break;
        case LEB_MODEL_PLANAR_QUAD: M.n = 6; M.N = 8; break;
        case LEB_MODEL_SATELLITE: M.n = 7; M.N = 10; break;
        default: M.n = 12 * M.n_units; M.N = 16 * M.n_units; break;
    }
    // derived constants: evaluated in FP64 from the FP32 parameters, rounded once to FP32
    const double dt = m.dt;
    M.dt = (float)dt;
    M.half_dt = (float)(0.5 * dt);
    M.dt6 = (float)(dt / 6.0);
    if (m.model_id == LEB_MODEL_PLANAR_QUAD) {
        M.inv_m = (float)(1.0 / (double)m.mass);
        M.g = m.g;
        M.k1 = (float)((double)m.k1 / (double)m.Jx);      // arm length / moment of inertia
    } else if (m.model_id != LEB_MODEL_UNICYCLE) {
        M.inv_m = (float)(1.0 / (double)m.mass);
        M.g = m.g;
        M.cp = (float)(((double)m.Jy - (double)m.Jz) / (double)m.Jx);
        M.cq = (float)(((double)m.Jz - (double)m.Jx) / (double)m.Jy);
        M.cr = (float)(((double)m.Jx - (double)m.Jy) / (double)m.Jz);
        M.iJx = (float)(1.0 / (double)m.Jx);
        M.iJy = (float)(1.0 / (double)m.Jy);
        M.iJz = (float)(1.0 / (double)m.Jz);
        M.k1 = m.k1;
        M.k3 = m.k3;
    }
    return M;
}

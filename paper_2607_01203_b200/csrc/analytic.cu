// analytic.cu -- leb_analytic_fwd / leb_vjp(kind 0): path-based interval-Hessian bound
// (Thm 1, eq. (15)) and its VJP, FP32 with directed rounding.
//
// Launch shape: one CTA per (tile, centre unit).  A tile is one (trajectory, timestep); a "unit"
// is one quadrotor of the chain (1 for unicycle / quad12).  The CTA's work items are the pairs
// (j <= k) of variables in the dependency cone of the unit; each thread evaluates, for its items,
// the second-order interval jets of the unit's outputs over the prefix box A^(j) (steps A1-A2 of
// SURVEY 8(a)) and folds H_kj D_j D_k into per-output partial sums (A3), which are combined by
// directed-rounding warp shuffles.  Nothing but the 2N inputs and 2n outputs of a tile touches HBM.
#include "an_core.cuh"
#include "internal.h"

namespace leb_an {

constexpr int kThreads = 128;
constexpr int kMaxVars = 64;

__device__ __forceinline__ float shfl_add_dn(float v, int off) { return __fadd_rd(v, __shfl_xor_sync(0xffffffffu, v, off)); }
__device__ __forceinline__ float shfl_add_up(float v, int off) { return __fadd_ru(v, __shfl_xor_sync(0xffffffffu, v, off)); }

// loads the tile's nominal point and radii into shared memory and validates them
__device__ bool load_tile(const float* __restrict__ nom, const float* __restrict__ rad, int N, float* nom_s, float* rad_s) {
    int bad = 0;
    for (int g = threadIdx.x; g < N; g += blockDim.x) {
        float a = nom[g], s = rad[g];
        nom_s[g] = a;
        rad_s[g] = s;
        if (!(fabsf(a) <= 3.0e38f) || !(s >= 0.f) || !(s <= 3.0e38f)) bad = 1;
    }
    return __syncthreads_or(bad) != 0;
}

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
template <int NOUT, bool UNICYCLE>
__global__ void __launch_bounds__(kThreads)
analytic_fwd_kernel(Model M, const float* __restrict__ nom, const float* __restrict__ rad, int ld_in,
                    float* __restrict__ r_lo, float* __restrict__ r_hi, int ld_out, int* __restrict__ domain_flag) {
    extern __shared__ float smem[];
    float* nom_s = smem;
    float* rad_s = smem + M.N;
    __shared__ int vars[kMaxVars];
    __shared__ int nvars;
    __shared__ float red_lo[kThreads / 32][NOUT], red_hi[kThreads / 32][NOUT];

    const int tile = blockIdx.y, unit = blockIdx.x;
    bool bad = load_tile(nom + (size_t)tile * ld_in, rad + (size_t)tile * ld_in, M.N, nom_s, rad_s);
    if (threadIdx.x == 0) {
        if (UNICYCLE) { for (int g = 0; g < 5; ++g) vars[g] = g; nvars = 5; }
        else nvars = window_vars(M, unit, vars);
    }
    __syncthreads();
    const int L = nvars, nitems = L * (L + 1) / 2;

    Iv<float> R[NOUT];
#pragma unroll
    for (int l = 0; l < NOUT; ++l) R[l] = iconst<float>(0.f);
    bool dom = false;
    if (!bad) {
        for (int t = threadIdx.x; t < nitems; t += blockDim.x) {
            int a, b;
            item_decode(t, L, &a, &b);
            Inputs<float> in{nom_s, rad_s, vars[a], vars[b]};
            Jet<float> f[NOUT];
            if (UNICYCLE) unicycle_f(M, in, f);
            else chain_center_f(M, in, unit, f, &dom);
#pragma unroll
            for (int l = 0; l < NOUT; ++l)
                R[l] = iadd(R[l], item_term(f[l].wjk, rad_s[in.j], rad_s[in.k], in.j == in.k));
        }
    }
    bad = (__syncthreads_or((int)dom) != 0) || bad;
    // directed-rounding reduction: lanes -> warps -> thread l
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int l = 0; l < NOUT; ++l) {
        float lo = R[l].lo, hi = R[l].hi;
#pragma unroll
        for (int off = 16; off; off >>= 1) { lo = shfl_add_dn(lo, off); hi = shfl_add_up(hi, off); }
        if (lane == 0) { red_lo[warp][l] = lo; red_hi[warp][l] = hi; }
    }
    __syncthreads();
    if (threadIdx.x < NOUT) {
        float lo = red_lo[0][threadIdx.x], hi = red_hi[0][threadIdx.x];
        for (int w = 1; w < kThreads / 32; ++w) { lo = __fadd_rd(lo, red_lo[w][threadIdx.x]); hi = __fadd_ru(hi, red_hi[w][threadIdx.x]); }
        if (bad) { lo = -INFINITY; hi = INFINITY; }
        size_t o = (size_t)tile * ld_out + (size_t)unit * NOUT + threadIdx.x;
        r_lo[o] = lo;
        r_hi[o] = hi;
    }
    if (bad && threadIdx.x == 0) atomicExch(domain_flag, 1);
}

// ---------------------------------------------------------------------------------------------
// VJP by forward-mode duals: work unit = (item, direction); direction = (window variable, nom|rad)
// ---------------------------------------------------------------------------------------------
struct DuArr {   // presents a float array as duals with a unit tangent at one index
    const float* a;
    int seed;
    __device__ __forceinline__ Du operator[](int g) const { return Du{a[g], g == seed ? 1.f : 0.f}; }
};
template <> struct Inputs<Du> {
    DuArr nom, rad;
    int j, k;
    __device__ __forceinline__ Jet<Du> operator()(int g) const {
        Jet<Du> r;
        if (g <= j) r.w = {add_dn(nom[g], neg(rad[g])), add_up(nom[g], rad[g])};
        else r.w = {nom[g], nom[g]};
        r.wj = iconst<Du>(g == j ? 1.f : 0.f);
        r.wk = iconst<Du>(g == k ? 1.f : 0.f);
        r.wjk = iconst<Du>(0.f);
        return r;
    }
};

template <int NOUT, bool UNICYCLE>
__global__ void __launch_bounds__(kThreads)
analytic_vjp_kernel(Model M, const float* __restrict__ nom, const float* __restrict__ rad,
                    const float* __restrict__ g_lo, const float* __restrict__ g_hi, int ld_in, int ld_out,
                    float* __restrict__ grad_nom, float* __restrict__ grad_rad, int* __restrict__ domain_flag) {
    extern __shared__ float smem[];
    float* nom_s = smem;
    float* rad_s = smem + M.N;
    __shared__ int vars[kMaxVars];
    __shared__ int nvars;
    __shared__ float gl_s[NOUT], gh_s[NOUT];
    __shared__ float grad_s[2 * kMaxVars];
    __shared__ int rad_off[kMaxVars + 1];      // prefix counts of the radius work units per item row a

    const int tile = blockIdx.y, unit = blockIdx.x;
    bool bad = load_tile(nom + (size_t)tile * ld_in, rad + (size_t)tile * ld_in, M.N, nom_s, rad_s);
    if (threadIdx.x == 0) {
        if (UNICYCLE) { for (int g = 0; g < 5; ++g) vars[g] = g; nvars = 5; }
        else nvars = window_vars(M, unit, vars);
    }
    if (threadIdx.x < NOUT) {
        size_t o = (size_t)tile * ld_out + (size_t)unit * NOUT + threadIdx.x;
        gl_s[threadIdx.x] = g_lo[o];
        gh_s[threadIdx.x] = g_hi[o];
    }
    for (int d = threadIdx.x; d < 2 * kMaxVars; d += blockDim.x) grad_s[d] = 0.f;
    __syncthreads();
    const int L = nvars, nitems = L * (L + 1) / 2, ndirs = 2 * L;
    // Work units.  Every item (a <= b) needs all L nominal directions.  A RADIUS direction p matters only if the box of the
    // item depends on sigma_p -- positions p <= a of the prefix box A^(j) (Thm 1: coordinates after j are pinned at the
    // nominal point, L162) -- or if sigma_p is one of the explicit factors (p == b; p == a is already counted): for every
    // other p the tangent is identically zero, so those (item, direction) pairs are not enumerated at all
    // (L = 54: 109 341 units instead of 160 380).  Row a of the item table has L - a items, each with a + 1 box directions.
    if (threadIdx.x == 0) {
        int acc = 0;
        for (int a = 0; a < L; ++a) { rad_off[a] = acc; acc += (L - a) * (a + 1); }
        rad_off[L] = acc;
    }
    __syncthreads();
    const int n_nom = nitems * L, n_box = rad_off[L], n_fac = nitems - L;      // n_fac: off-diagonal items, direction p == b
    bool dom = false;
    if (!bad) {
        const int nwork = n_nom + n_box + n_fac;
        for (int w = threadIdx.x; w < nwork; w += blockDim.x) {
            int a, b, d;                       // item (a, b) and direction d in [0, 2L): nominal d, radius L + position
            if (w < n_nom) {
                const int t = w / L;
                d = w - t * L;
                item_decode(t, L, &a, &b);
            } else if (w < n_nom + n_box) {
                const int r = w - n_nom;
                int lo = 0, hi = L - 1;        // largest a with rad_off[a] <= r
                while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (rad_off[mid] <= r) lo = mid; else hi = mid - 1; }
                a = lo;
                const int rem = r - rad_off[a], p = rem / (L - a);
                b = a + (rem - p * (L - a));
                d = L + p;
            } else {
                item_decode_offdiag(w - n_nom - n_box, L, &a, &b);
                d = L + b;
            }
            const int j = vars[a], k = vars[b];
            const int dvar = vars[d < L ? d : d - L];
            Inputs<Du> in{DuArr{nom_s, d < L ? dvar : -1}, DuArr{rad_s, d < L ? -1 : dvar}, j, k};
            Jet<Du> f[NOUT];
            if (UNICYCLE) unicycle_f(M, in, f);
            else chain_center_f(M, in, unit, f, &dom);
            float acc = 0.f;
#pragma unroll
            for (int l = 0; l < NOUT; ++l) {
                Iv<Du> term = item_term(f[l].wjk, in.rad[j], in.rad[k], j == k);
                acc = fmaf(gh_s[l], term.hi.d, acc);
                acc = fmaf(gl_s[l], term.lo.d, acc);
            }
            atomicAdd(&grad_s[d], acc);
        }
    }
    bad = (__syncthreads_or((int)dom) != 0) || bad;
    for (int d = threadIdx.x; d < ndirs; d += blockDim.x) {
        float v = bad ? NAN : grad_s[d];
        int var = vars[d < L ? d : d - L];
        float* dst = (d < L ? grad_nom : grad_rad) + (size_t)tile * ld_in + var;
        atomicAdd(dst, v);
    }
    if (bad && threadIdx.x == 0) atomicExch(domain_flag, 1);
}

// zero the first N columns of [tiles, ld] rows
__global__ void zero_rows_kernel(float* __restrict__ a, float* __restrict__ b, int tiles, int N, int ld) {
    size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t total = (size_t)tiles * N;
    if (idx < total) {
        size_t t = idx / N, c = idx - t * N;
        a[t * ld + c] = 0.f;
        b[t * ld + c] = 0.f;
    }
}

}  // namespace leb_an

using namespace leb_an;

Model leb_make_model(const leb_analytic_model& m) {
    Model M{};
    M.id = m.model_id;
    M.integ = (m.model_id == LEB_MODEL_UNICYCLE) ? LEB_INTEG_EULER : m.integ;
    M.n_units = (m.model_id == LEB_MODEL_QUADCHAIN) ? m.n_units : 1;
    if (m.model_id == LEB_MODEL_UNICYCLE) { M.n = 3; M.N = 5; }
    else { M.n = 12 * M.n_units; M.N = 16 * M.n_units; }
    // derived constants: evaluated in FP64 from the FP32 parameters, rounded once to FP32
    double dt = m.dt;
    M.dt = (float)dt;
    M.half_dt = (float)(0.5 * dt);
    M.dt6 = (float)(dt / 6.0);
    if (m.model_id != LEB_MODEL_UNICYCLE) {
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

cudaError_t leb_launch_analytic_fwd(const Model& M, int tiles, const float* nom, const float* rad, int ld_in,
                                    float* r_lo, float* r_hi, int ld_out, int* domain_flag, cudaStream_t st,
                                    long long* launches, LebProf* prof) {
    if (tiles == 0) return cudaSuccess;
    size_t smem = 2 * (size_t)M.N * sizeof(float);
    // gridDim.y is limited to 65535: slice the tile range
    for (int t0 = 0; t0 < tiles; t0 += 65535) {
        int nt = tiles - t0 < 65535 ? tiles - t0 : 65535;
        const float* a = nom + (size_t)t0 * ld_in;
        const float* s = rad + (size_t)t0 * ld_in;
        float* lo = r_lo + (size_t)t0 * ld_out;
        float* hi = r_hi + (size_t)t0 * ld_out;
        prof->begin(LEB_KC_ANALYTIC_FWD, st);
        if (M.id == LEB_MODEL_UNICYCLE)
            analytic_fwd_kernel<3, true><<<dim3(1, nt), kThreads, smem, st>>>(M, a, s, ld_in, lo, hi, ld_out, domain_flag);
        else
            analytic_fwd_kernel<12, false><<<dim3(M.n_units, nt), kThreads, smem, st>>>(M, a, s, ld_in, lo, hi, ld_out, domain_flag);
        prof->end(LEB_KC_ANALYTIC_FWD, st, 0.0);
        ++*launches;
    }
    return cudaGetLastError();
}

cudaError_t leb_launch_analytic_vjp(const Model& M, int tiles, const float* nom, const float* rad, const float* g_lo,
                                    const float* g_hi, int ld_in, int ld_out, float* grad_nom, float* grad_rad,
                                    int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof) {
    if (tiles == 0) return cudaSuccess;
    size_t smem = 2 * (size_t)M.N * sizeof(float);
    size_t total = (size_t)tiles * M.N;
    zero_rows_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(grad_nom, grad_rad, tiles, M.N, ld_in);
    ++*launches;
    for (int t0 = 0; t0 < tiles; t0 += 65535) {
        int nt = tiles - t0 < 65535 ? tiles - t0 : 65535;
        size_t oi = (size_t)t0 * ld_in, oo = (size_t)t0 * ld_out;
        prof->begin(LEB_KC_ANALYTIC_VJP, st);
        if (M.id == LEB_MODEL_UNICYCLE)
            analytic_vjp_kernel<3, true><<<dim3(1, nt), kThreads, smem, st>>>(M, nom + oi, rad + oi, g_lo + oo, g_hi + oo, ld_in,
                                                                             ld_out, grad_nom + oi, grad_rad + oi, domain_flag);
        else
            analytic_vjp_kernel<12, false><<<dim3(M.n_units, nt), kThreads, smem, st>>>(M, nom + oi, rad + oi, g_lo + oo, g_hi + oo,
                                                                                       ld_in, ld_out, grad_nom + oi, grad_rad + oi,
                                                                                       domain_flag);
        prof->end(LEB_KC_ANALYTIC_VJP, st, 0.0);
        ++*launches;
    }
    return cudaGetLastError();
}

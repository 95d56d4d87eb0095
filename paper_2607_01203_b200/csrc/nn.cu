// nn.cu -- leb_nn_fwd / leb_vjp(kind 1): CROWN back-substitution (Thm 2, eq. (18),
// PAPER.md:L196-200) + Jacobian correction and box concretisation (Thm 3, eq. (19)-(21), L204-220),
// and the reverse sweep of the same computation.
//
// Formulation ("deviation form"; algebraically identical to eq. (18)-(21), SURVEY
// 8(c).7): with zhat_l the nominal pre-activations and, per neuron, the gaps
// gU = kU zhat + bU - phi(zhat) >= 0, gL = kL zhat + bL - phi(zhat) <= 0 of the two relaxation lines,
//     u_s = zhat_s + |Lam_up_0| sigma + sum_l (P_l gU_l + Q_l gL_l)          (hidden target s)
//     l_s = zhat_s - |Lam_lo_0| sigma + sum_l (P_l gL_l + Q_l gU_l)
//     r_hi = |Lam_up_0 - J| sigma + sum_l (...),  r_lo = -|Lam_lo_0 - J| sigma + sum_l (...)   (output)
// where Lam_{l-1} = (P_l (.) k_pos + Q_l (.) k_neg) W_l, P = max(Lam,0), Q = min(Lam,0), and J is the
// third ("Jacobian") chain with k_pos = k_neg = phi'(zhat).  No O(1) quantities are cancelled.
//
// Steps: N1 nominal pass, N2 layer-1 interval bounds, N3 hidden targets, N4 output
// target, N5 concretisation, V reverse sweep.  All contractions are launched from here.
#include <stdio.h>
#include <stdlib.h>
#include <vector>
#include "internal.h"
#include "nn_relax.cuh"
#include "nn_gemm_ffma.cuh"
#include "nn_gemm_tc.cuh"
#include "nn_gemm_tc2.cuh"

using namespace leb_nn;

namespace {

inline int rup(int x, int m) { return (x + m - 1) / m * m; }
constexpr int kPad = 32;        // feature dims are zero-padded to multiples of 32
constexpr int kRowBlock = 256;  // chain row blocks (the tensor-core kernel takes 256 coefficient rows per tile)
constexpr int kMaxLayers = 16;

}  // namespace

struct NnState {
    bool ready = false;
    int L = 0, act = 0;
    int w[kMaxLayers + 1] = {0}, wp[kMaxLayers + 1] = {0};   // true / padded widths, w[0] = N, w[L] = n
    // weights (1-based layer index l = 1..L): W[l] is [rowsW[l] x wp[l-1]], Wt[l] is [wp[l-1] x rowsW[l]]
    float *W[kMaxLayers + 1] = {nullptr}, *Wt[kMaxLayers + 1] = {nullptr}, *bias[kMaxLayers + 1] = {nullptr};
    int rowsW[kMaxLayers + 1] = {0};
    float *Wabs1 = nullptr, *Wabs1t = nullptr;
    float *Wabs[kMaxLayers + 1] = {nullptr}, *Wabst[kMaxLayers + 1] = {nullptr};   // |W_l|, |W_l|^T for l = 2..L-1 (CROWN-IBP mode)
    // 3xTF32 tensor-core path: hi/lo splits of W[l] (reverse sweep) and Wt[l] (forward chain), l = 1..L-1, and their TMA maps
    float *Whi[kMaxLayers + 1] = {nullptr}, *Wlo[kMaxLayers + 1] = {nullptr}, *Wthi[kMaxLayers + 1] = {nullptr}, *Wtlo[kMaxLayers + 1] = {nullptr};
    CUtensorMap mapW_hi[kMaxLayers + 1], mapW_lo[kMaxLayers + 1], mapWt_hi[kMaxLayers + 1], mapWt_lo[kMaxLayers + 1];
    bool tc_ready = false, use_tc = false, launch_failed = false;
    bool use_pairs = false;      // forward chain steps on CTA pairs (nn_gemm_tc2.cuh)
    int num_sms = 148;
    // workspace for one chunk of tiles
    int chunk_req = 0, chunk = 0;
    bool chunk_capped = false;   // the default chunk was limited by free memory
    bool ws_vjp = false;
    std::vector<void*> allocs;
    float *nomp = nullptr, *radp = nullptr, *rad1 = nullptr;
    float *mup = nullptr, *mu1 = nullptr, *mu_bar = nullptr;   // non-centred boxes: padded mu, W_1 mu, and its adjoint
    float *ibp_c = nullptr, *ibp_r = nullptr, *ibp_a = nullptr, *ibp_m = nullptr, *ibp_vm = nullptr;   // certified CROWN-IBP scratch
    float* alpha[kMaxLayers] = {nullptr};                      // optimisable lower ReLU slopes (leb_nn_alpha_fwd), [chunk x wp[l]]
    float* alpha_best[kMaxLayers] = {nullptr};                 // ... of the tightest iterate so far
    int* alpha_take = nullptr;                                 // [chunk]: did the last iterate improve the tile?
    bool last_alpha = false;                                   // the resident forward state was computed with refined slopes
    int alpha_mode = 0;                                        // 0 off, 1 forward writes the adaptive default, 2 forward reads alpha
    std::vector<void*> alpha_scratch; size_t alpha_scratch_tiles = 0;
    const float* mu_cur = nullptr;                             // = mup while the chunk in flight has box offsets, else NULL
    float *zhat[kMaxLayers] = {nullptr}, *ahat[kMaxLayers] = {nullptr}, *dphi[kMaxLayers] = {nullptr};
    float *lb[kMaxLayers] = {nullptr}, *ub[kMaxLayers] = {nullptr};
    float *kU[kMaxLayers] = {nullptr}, *kL[kMaxLayers] = {nullptr}, *gU[kMaxLayers] = {nullptr}, *gL[kMaxLayers] = {nullptr};
    // chains: target s = 2..L; Lam[s][l] for l = 0..s-2: [chunk*rows_pad[s] x wp[l]]
    int rows_kind[kMaxLayers + 1] = {0}, rows_pad[kMaxLayers + 1] = {0};
    float* Lam[kMaxLayers + 1][kMaxLayers] = {{nullptr}};
    float* gap[kMaxLayers + 1] = {nullptr};
    // certified mode (N6, DESIGN.md §6 "Certified margin"): per layer the centre residual e, the nominal drift t, the
    // interval radius v of z_l - zhat_l, the activation deviation adev and the gap pads mU, mL ([chunk x wp[l]]);
    // the chain margin of the output rows (report only, [chunk x rows_pad[L]]); eta for the output ([chunk x wpL])
    float *ce[kMaxLayers] = {nullptr}, *ct[kMaxLayers] = {nullptr}, *cv[kMaxLayers] = {nullptr}, *adev[kMaxLayers] = {nullptr};
    float *mU[kMaxLayers] = {nullptr}, *mL[kMaxLayers] = {nullptr}, *marg = nullptr, *eta = nullptr;
    // VJP workspace
    float *kUb[kMaxLayers] = {nullptr}, *kLb[kMaxLayers] = {nullptr}, *gUb[kMaxLayers] = {nullptr}, *gLb[kMaxLayers] = {nullptr},
          *dpb[kMaxLayers] = {nullptr}, *zbar[kMaxLayers] = {nullptr}, *lbar[kMaxLayers] = {nullptr}, *ubar[kMaxLayers] = {nullptr};
    float *Lbar[2] = {nullptr, nullptr}, *gapbar = nullptr, *nom_bar = nullptr, *rad_bar = nullptr, *glo_p = nullptr, *ghi_p = nullptr;
    int last_tiles = 0;          // > 0: the workspace holds the complete forward state of that many tiles (one chunk)
    bool last_with_jac = false;  // ... including the Jacobian chain rows (needed by the reverse sweep)
    bool last_cert = false;      // ... computed in certified mode (widened hidden bounds, padded gaps)
    bool last_ibp = false;       // ... with hidden-layer bounds by interval propagation (LEB_FLAG_IBP_HIDDEN)
    bool last_mu = false;        // ... on non-centred boxes (mu != NULL)
    bool last_vjp_reused = false;   // the last leb_vjp(kind 1) started from the resident forward state
    LebProf* prof = nullptr;
};

namespace {

// ------------------------------------------------------------------------------------------
// small kernels
// ------------------------------------------------------------------------------------------
// copy [rows x cols] (ld_src) into a zero-padded [rows x ld_dst] buffer, optionally transposing / abs
__global__ void pack_matrix_kernel(const float* __restrict__ src, int rows, int cols, int ld_src, float* __restrict__ dst,
                                   int rows_p, int cols_p, int transpose, int absval) {
    // dst is [rows_p x cols_p] if !transpose else [cols_p x rows_p]
    size_t total = (size_t)rows_p * cols_p;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int r, c;
        if (!transpose) { r = (int)(q / cols_p); c = (int)(q - (size_t)r * cols_p); }
        else { c = (int)(q / rows_p); r = (int)(q - (size_t)c * rows_p); }
        float v = (r < rows && c < cols) ? src[(size_t)r * ld_src + c] : 0.f;
        dst[q] = absval ? fabsf(v) : v;
    }
}

// nom/rad [tiles x ld_in] -> zero-padded [tiles x wp0]; invalid input (NaN/Inf, sigma < 0) poisons the tile with NaN
__global__ void pad_inputs_kernel(int tiles, int N, int ld_in, int wp0, const float* __restrict__ nom, const float* __restrict__ rad,
                                  float* __restrict__ nomp, float* __restrict__ radp, const float* __restrict__ mu = nullptr,
                                  float* __restrict__ mup = nullptr) {
    size_t total = (size_t)tiles * wp0;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(q / wp0), c = (int)(q - (size_t)t * wp0);
        float a = 0.f, s = 0.f;
        if (c < N) {
            a = nom[(size_t)t * ld_in + c];
            s = rad[(size_t)t * ld_in + c];
            if (!(s >= 0.f) || !(s <= 3.0e38f)) s = NAN;
            if (!(fabsf(a) <= 3.0e38f)) a = NAN;
        }
        nomp[q] = a;
        radp[q] = s;
        if (mup) {
            float m = (c < N) ? mu[(size_t)t * ld_in + c] : 0.f;
            if (!(fabsf(m) <= 3.0e38f)) m = NAN;
            mup[q] = m;
        }
    }
}

__global__ void pad_cotangent_kernel(int tiles, int n, int ld_out, const float* __restrict__ g_lo, const float* __restrict__ g_hi,
                                     float* __restrict__ glo_p, float* __restrict__ ghi_p) {
    size_t total = (size_t)tiles * n;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(q / n), c = (int)(q - (size_t)t * n);
        glo_p[q] = g_lo[(size_t)t * ld_out + c];
        ghi_p[q] = g_hi[(size_t)t * ld_out + c];
    }
}

__global__ void fill_kernel(float* __restrict__ p, size_t count, float v) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x) p[q] = v;
}

// x = hi + lo with hi = tf32(x), lo = tf32(x - hi) (round to nearest, ties away): operands of the 3xTF32 contraction
__global__ void split_tf32_kernel(const float* __restrict__ src, float* __restrict__ hi, float* __restrict__ lo, size_t count) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x) {
        const float x = src[q], h = tc::to_tf32(x);
        hi[q] = h;
        lo[q] = tc::to_tf32(x - h);
    }
}

// per-neuron relaxation of layer l from (zhat, l, u); for layer 1 (rad1 != NULL) first l,u = zhat -+ rad1 (N2)
__global__ void relax_fwd_kernel(int act, int tiles, int w_valid, int wp, const float* __restrict__ zhat,
                                 const float* __restrict__ rad1, float* __restrict__ lb, float* __restrict__ ub,
                                 float* __restrict__ kU, float* __restrict__ kL, float* __restrict__ gU, float* __restrict__ gL,
                                 const float* __restrict__ mu1 = nullptr, float* __restrict__ alpha = nullptr, int alpha_mode = 0) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) {
            lb[q] = 0.f; ub[q] = 0.f; kU[q] = 0.f; kL[q] = 0.f; gU[q] = 0.f; gL[q] = 0.f;
            continue;
        }
        float z = zhat[q], l, u;
        if (rad1) {     // layer 1: z_1 - zhat_1 = W_1 (a - a~) in W_1 mu -+ |W_1| sigma   (mu1 = W_1 mu, non-centred boxes)
            const float r = rad1[q], m = mu1 ? mu1[q] : 0.f;
            l = z + (m - r); u = z + (m + r); lb[q] = l; ub[q] = u;
        }
        else { l = lb[q]; u = ub[q]; }
        Relax r = relax_any(act, (double)l, (double)u);
        if (alpha_mode) {     // optimisable lower slope of an unstable ReLU neuron: any value in [0, 1] is a valid lower line
            if (alpha_mode == 1) alpha[q] = (float)r.kL;
            else if (r.cL == LINE_RELU_LOW) r.kL = (double)alpha[q];
        }
        double f = act_f(act, (double)z);
        kU[q] = (float)r.kU;
        kL[q] = (float)r.kL;
        gU[q] = (float)(r.kU * (double)z + r.bU - f);
        gL[q] = (float)(r.kL * (double)z + r.bL - f);
    }
}

// certified mode (N6): the same relaxation, made sound for the numbers as STORED.  With c = zhat (the FP32 centre),
// a = ahat (the FP32 centre of the activation) and the FP32 slopes kU, kL, the stored gaps satisfy, for every z in [l, u],
//     kL (z - c) + gL  <=  phi(z) - a  <=  kU (z - c) + gU            in exact arithmetic:
// the slope's rounding moves the line by at most |k32 - k64| max|z - c|, and the FP64 construction of the line by at most
// d64 (libm tanh within 2 ulp); both are added outward, gU is rounded up and kept >= 0, gL rounded down and kept <= 0.
// Layer 1 (layer1 != 0): l, u = c -+ (|W_1| sigma + e_1) = c -+ (v + e), outward.  adev >= |phi(z) - a| over [l, u].
//
// The rounding of the chain step through this layer is carried by the gaps as well.  A coefficient row Lam on a_l turns
// into D = Lam^+ kU + Lam^- kL (lower chain: kL, kU) and then into D W_l, computed in FP32 / 3xTF32; what the step can lose
// is at most sum_j |D_j| x_j with x_j = gamma_j v_j + e_j (v = |W_l| adev_{l-1}: radius of z_l - zhat_l; e: centre residual;
// gamma_j: see gamma_of()), and |D_j| x_j = Lam_j^+ |kU_j| x_j - Lam_j^- |kL_j| x_j has exactly the form of the gap sum.  So
//     gU += |kU| x,   gL -= |kL| x
// adds the step's margin outward to both chains, on either contraction path, with no work in the contraction kernels.
// mU, mL keep the two pads by themselves (for the margin report).
__device__ __forceinline__ float gamma_of(int tensor, int K, int j) {
    // rounding error that the product D_j W_l[j,k] can cause in the contraction over j (K terms, taken in index order by
    // both kernels): the term is part of every partial sum from its own step on.
    //   tensor path: (4.5 (K/8 - floor(j/8)) + 17) 2^-23 -- per accumulating MMA (8 terms) at most 4.5 ulp of the running
    //                magnitude (measured adder: addends truncated at 2^-25 of the largest, result truncated to FP32; taken
    //                twice over in case the 8 terms are added in two halves), + 2^-19 for the hi/lo split, the dropped
    //                lo*lo term and the correction accumulator, + 2^-23 for the rounding of D_j itself and the final FADD
    //   FFMA path:   (K - j + 4) 2^-24 + 2^-23         -- one rounding to nearest per fused multiply-add
    // (DESIGN.md section 6 "Certified margin"; tests/test_gpu_nn_certified.py probes both models on adversarial operands)
    const float g = tensor ? (4.5f * (float)(K / 8 - j / 8) + 17.f) * 1.1920930e-07f : (float)(K - j + 4) * 5.9604652e-08f + 1.1920930e-07f;
    return g * 1.000001f;
}
__global__ void relax_fwd_cert_kernel(int act, int tiles, int w_valid, int wp, int layer1, int tensor, const float* __restrict__ zhat,
                                      const float* __restrict__ ahat, const float* __restrict__ v, const float* __restrict__ e,
                                      float* __restrict__ lb, float* __restrict__ ub, float* __restrict__ kU, float* __restrict__ kL,
                                      float* __restrict__ gU, float* __restrict__ gL, float* __restrict__ adev,
                                      float* __restrict__ mU, float* __restrict__ mL, const float* __restrict__ m1 = nullptr,
                                      const float* __restrict__ vmu = nullptr, float gam_mu = 0.f,
                                      const float* __restrict__ alpha = nullptr) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) {
            lb[q] = 0.f; ub[q] = 0.f; kU[q] = 0.f; kL[q] = 0.f; gU[q] = 0.f; gL[q] = 0.f; adev[q] = 0.f; mU[q] = 0.f; mL[q] = 0.f;
            continue;
        }
        float z = zhat[q], l, u;
        float vq = v[q];          // radius of z - zhat over the box (what the rounding pads below scale with)
        if (layer1) {
            float r = __fadd_ru(vq, e[q]);
            if (m1) {
                // non-centred box: z_1 - zhat_1 in W_1 mu -+ |W_1| sigma -+ e_1.  m1 is the FP32 product W_1 mu, wrong by at
                // most gam_mu |W_1||mu| (vmu, rounded up); the radius seen by the pads is |W_1| (sigma + |mu|)
                const float mq = m1[q];
                r = __fadd_ru(r, __fmul_ru(gam_mu, vmu[q]));
                l = __fadd_rd(z, __fadd_rd(mq, -r)); u = __fadd_ru(z, __fadd_ru(mq, r));
                vq = __fadd_ru(vq, vmu[q]);
            } else {
                l = __fadd_rd(z, -r); u = __fadd_ru(z, r);
            }
            lb[q] = l; ub[q] = u;
        } else { l = lb[q]; u = ub[q]; }
        const double zd = (double)z, ld = (double)l, ud = (double)u, a = (double)ahat[q];
        Relax r = relax_any(act, ld, ud);
        if (alpha && r.cL == LINE_RELU_LOW) r.kL = (double)alpha[q];      // a given lower slope in [0, 1]: as sound as the rule's
        const float kU32 = (float)r.kU, kL32 = (float)r.kL;
        const double zdev = fmax(ud - zd, zd - ld);
        const double d64 = 5.7e-14 * (1.0 + fabs(zd) + fabs(ld) + fabs(ud));          // 2^-44 (1 + |c| + |l| + |u|)
        const double gu = (r.kU * zd + r.bU - a) + fabs((double)kU32 - r.kU) * zdev + d64;
        const double gl = (r.kL * zd + r.bL - a) - fabs((double)kL32 - r.kL) * zdev - d64;
        const float x = __fmaf_ru(gamma_of(tensor, wp, c), vq, e[q]);
        const float pu = __fmul_ru(fabsf(kU32), x), pl = __fmul_ru(fabsf(kL32), x);
        kU[q] = kU32;
        kL[q] = kL32;
        gU[q] = __fadd_ru(fmaxf(__double2float_ru(gu), 0.f), pu);
        gL[q] = __fadd_rd(fminf(__double2float_rd(gl), 0.f), -pl);
        mU[q] = pu;
        mL[q] = pl;
        adev[q] = __double2float_ru(fmax(act_f(act, ud) - a, a - act_f(act, ld)) + 1e-15);
    }
}

// certified mode (N6): one layer's rounding bookkeeping from the stored centres.  For tile m and neuron j of layer l,
//   e[m,j] >= | W_l ahat_{l-1} + b_l - zhat_l |      FP64 dot product (a product of two floats is exact in FP64) + its own
//                                                     accumulation bound (K + 2) 2^-52 (|W_l| |ahat_{l-1}| + |b_l|)
//   t[m,j] >= | a_l(nominal input) - ahat_l |         = (|W_l| t_{l-1} + e) + |phi(zhat_l) - ahat_l|   (phi is 1-Lipschitz)
//   v[m,j] >= |W_l| adev_{l-1}                        radius of z_l - zhat_l - (centre residual) over the box
// the two |W_l| products are FP32 with every operation rounded up.  out_only (layer L): t = eta = |W_L| t_{L-1}.
// Wt is [K x ldw] (K-major: Wt[k][j]).  Block: 16 tiles x 64 neurons, K slabs of 32.
constexpr int CM = 16, CJ = 64, CK = 32;
__global__ void __launch_bounds__(256) cert_layer_kernel(int C, int J, int K, const float* __restrict__ Wt, int ldw,
                                                         const float* __restrict__ bias, const float* __restrict__ X,
                                                         const float* __restrict__ T, const float* __restrict__ A, int ldx,
                                                         const float* __restrict__ zhat, const float* __restrict__ ahat, int act,
                                                         int out_only, float* __restrict__ e, float* __restrict__ t,
                                                         float* __restrict__ v, int ldo) {
    // weights and centres are converted to FP64 once per block load (a conversion per use made the kernel conversion-bound)
    __shared__ __align__(16) float Ws[CK][CJ];
    __shared__ __align__(16) double Wd[CK][CJ];
    __shared__ float Ts[CM][CK], As[CM][CK];
    __shared__ double Xd[CM][CK];
    const int tid = threadIdx.x, tj = tid & 15, tm = tid >> 4;
    const int m0 = blockIdx.y * CM, j0 = blockIdx.x * CJ;
    double s[4] = {0.0, 0.0, 0.0, 0.0}, sa[4] = {0.0, 0.0, 0.0, 0.0};
    float zt[4] = {0.f, 0.f, 0.f, 0.f}, vv[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k0 = 0; k0 < K; k0 += CK) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int idx = tid + i * 256, kk = idx >> 6, jj = idx & 63;
            const float wv = (k0 + kk < K && j0 + jj < J) ? Wt[(size_t)(k0 + kk) * ldw + j0 + jj] : 0.f;
            Ws[kk][jj] = fabsf(wv);
            Wd[kk][jj] = (double)wv;
        }
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int idx = tid + i * 256, mm = idx >> 5, kk = idx & 31;
            const bool ok = (m0 + mm < C) && (k0 + kk < K);
            const size_t o = (size_t)(m0 + mm) * ldx + k0 + kk;
            Xd[mm][kk] = (ok && X) ? (double)X[o] : 0.0;
            Ts[mm][kk] = (ok && T) ? T[o] : 0.f;
            As[mm][kk] = (ok && A) ? A[o] : 0.f;
        }
        __syncthreads();
#pragma unroll 4
        for (int kk = 0; kk < CK; ++kk) {
            const float4 w4 = *reinterpret_cast<const float4*>(&Ws[kk][tj * 4]);                 // |W|
            const float wabs[4] = {w4.x, w4.y, w4.z, w4.w};
            const double2 d01 = *reinterpret_cast<const double2*>(&Wd[kk][tj * 4]), d23 = *reinterpret_cast<const double2*>(&Wd[kk][tj * 4 + 2]);
            const double wd[4] = {d01.x, d01.y, d23.x, d23.y};
            const double x = Xd[tm][kk], xa = fabs(x);
            const float tt = Ts[tm][kk], a = As[tm][kk];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                if (!out_only) {
                    s[c] = fma(wd[c], x, s[c]);
                    sa[c] = fma(fabs(wd[c]), xa, sa[c]);
                    vv[c] = __fmaf_ru(wabs[c], a, vv[c]);
                }
                zt[c] = __fmaf_ru(wabs[c], tt, zt[c]);
            }
        }
        __syncthreads();
    }
    const int m = m0 + tm;
    if (m >= C) return;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int j = j0 + tj * 4 + c;
        if (j >= J) continue;
        const size_t o = (size_t)m * ldo + j;
        if (out_only) { t[o] = zt[c]; continue; }
        const double b = (double)bias[j], c0 = (double)zhat[o];
        const double fuzz = (sa[c] + fabs(b)) * (double)(K + 2) * 2.220446049250313e-16;
        const float ee = __double2float_ru(fabs(s[c] + b - c0) + fuzz);
        const double ep = fabs(act_f(act, c0) - (double)ahat[o]) + 1e-15;
        e[o] = ee;
        t[o] = __fadd_ru(__fadd_ru(zt[c], ee), __double2float_ru(ep));
        v[o] = vv[c];
    }
}

// certified mode, margin report: the share of the output rows' gap sums that is rounding pad,
//   marg[row] (+)= sum_j Lam_j^+ m_pos[j] - Lam_j^- m_neg[j]      (upper rows: (mU, mL); lower rows: (mL, mU))
// for one chain step of the output target; one warp per row (upper and lower rows only).  Rounded up.
__global__ void row_margin_kernel(int tiles, int rows_pad, int rows_kind, int K, const float* __restrict__ Lam, int a_shared,
                                  const float* __restrict__ mU, const float* __restrict__ mL, float* __restrict__ marg, int init) {
    int warp = (int)(((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (warp >= tiles * 2 * rows_kind) return;
    const int t = warp / (2 * rows_kind), r = warp - t * 2 * rows_kind, kind = r / rows_kind, rk = r - kind * rows_kind;
    const float* row = Lam + (size_t)(a_shared ? rk : (size_t)t * rows_pad + r) * K;
    const float* mp = (kind == 0 ? mU : mL) + (size_t)t * K;
    const float* mn = (kind == 0 ? mL : mU) + (size_t)t * K;
    float s = 0.f;
    for (int j = lane; j < K; j += 32) {
        const float lv = row[j];
        s = __fmaf_ru(fabsf(lv), lv > 0.f ? mp[j] : mn[j], s);
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) s = __fadd_ru(s, __shfl_xor_sync(0xffffffffu, s, off));
    if (lane == 0) marg[(size_t)t * rows_pad + r] = init ? s : __fadd_ru(marg[(size_t)t * rows_pad + r], s);
}

// N5 for a hidden target s: one warp per (tile, neuron k): rows k (upper) and rows_kind + k (lower)
// certified mode (e_s != NULL): every term rounded outward -- the |Lam| sigma sums and the gap sums (which carry the
// chain steps' rounding pads, see relax_fwd_cert_kernel) are sums of same-signed terms, so their FP32 rounding error is
// relative (factors kap_sum, kap_gap); plus the centre residual e_s of the target neuron (DESIGN.md §6 "Certified margin")
__global__ void concretise_hidden_kernel(int tiles, int rows_pad, int rows_kind, int wp0, const float* __restrict__ Lam0,
                                         const float* __restrict__ sigma, const float* __restrict__ gap,
                                         const float* __restrict__ zhat, float* __restrict__ lb, float* __restrict__ ub,
                                         const float* __restrict__ e_s, float kap_sum, float kap_gap,
                                         const float* __restrict__ mu = nullptr) {
    int warp = (int)(((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    int total = tiles * rows_kind;
    if (warp >= total) return;
    int t = warp / rows_kind, k = warp - t * rows_kind;
    const float* up = Lam0 + ((size_t)t * rows_pad + k) * wp0;
    const float* lo = Lam0 + ((size_t)t * rows_pad + rows_kind + k) * wp0;
    const float* sg = sigma + (size_t)t * wp0;
    float su = 0.f, sl = 0.f, du = 0.f, dl = 0.f;        // du, dl: Lam_0 mu (non-centred boxes: a - a~ in mu -+ sigma)
    float au = 0.f, al = 0.f;                            // |Lam_0| |mu|: what the rounding of du, dl scales with (certified mode)
    for (int j = lane * 4; j < wp0; j += 128) {
        float4 a = *reinterpret_cast<const float4*>(up + j), b = *reinterpret_cast<const float4*>(lo + j);
        float4 s = *reinterpret_cast<const float4*>(sg + j);
        su += fabsf(a.x) * s.x + fabsf(a.y) * s.y + fabsf(a.z) * s.z + fabsf(a.w) * s.w;
        sl += fabsf(b.x) * s.x + fabsf(b.y) * s.y + fabsf(b.z) * s.z + fabsf(b.w) * s.w;
        if (mu) {
            float4 m = *reinterpret_cast<const float4*>(mu + (size_t)t * wp0 + j);
            du += a.x * m.x + a.y * m.y + a.z * m.z + a.w * m.w;
            dl += b.x * m.x + b.y * m.y + b.z * m.z + b.w * m.w;
            au += fabsf(a.x * m.x) + fabsf(a.y * m.y) + fabsf(a.z * m.z) + fabsf(a.w * m.w);
            al += fabsf(b.x * m.x) + fabsf(b.y * m.y) + fabsf(b.z * m.z) + fabsf(b.w * m.w);
        }
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) {
        su += __shfl_xor_sync(0xffffffffu, su, off); sl += __shfl_xor_sync(0xffffffffu, sl, off);
        du += __shfl_xor_sync(0xffffffffu, du, off); dl += __shfl_xor_sync(0xffffffffu, dl, off);
        au += __shfl_xor_sync(0xffffffffu, au, off); al += __shfl_xor_sync(0xffffffffu, al, off);
    }
    if (lane == 0) {
        float z = zhat[(size_t)t * rows_kind + k];
        const float gu = gap[(size_t)t * rows_pad + k], gl = gap[(size_t)t * rows_pad + rows_kind + k];
        if (e_s) {
            const float e = e_s[(size_t)t * rows_kind + k];
            // the signed sums du, dl (non-centred boxes) are wrong by at most (wp0 + 8) 2^-24 of the sums of magnitudes
            const float km = __fmul_ru(__fadd_ru(kap_sum, -1.f), 1.0001f);      // (au, al are FP32 sums themselves)
            const float pu = __fadd_ru(__fadd_ru(__fadd_ru(__fmul_ru(su, kap_sum), __fmul_ru(gu, kap_gap)), e), __fadd_ru(du, __fmul_ru(au, km)));
            const float pl = __fadd_ru(__fadd_ru(__fadd_ru(__fmul_ru(sl, kap_sum), __fmul_ru(-gl, kap_gap)), e), __fadd_ru(-dl, __fmul_ru(al, km)));
            ub[(size_t)t * rows_kind + k] = __fadd_ru(z, pu);
            lb[(size_t)t * rows_kind + k] = __fadd_rd(z, -pl);
        } else {
            ub[(size_t)t * rows_kind + k] = z + ((su + du) + gu);
            lb[(size_t)t * rows_kind + k] = z - ((sl - dl) - gl);
        }
    }
}

// N5 for the output: Thm 3 (20)-(21); J = rows of the Jacobian chain, or the caller's matrix
__global__ void concretise_out_kernel(int tiles, int rows_pad, int n, int N, int wp0, const float* __restrict__ Lam0,
                                      const float* __restrict__ sigma, const float* __restrict__ gap,
                                      const float* __restrict__ Jgiven, float* __restrict__ r_lo, float* __restrict__ r_hi,
                                      int ld_out, int* __restrict__ domain_flag, int cert, const float* __restrict__ marg,
                                      const float* __restrict__ eta, int ld_eta, float kap_sum, float kap_gap,
                                      float* __restrict__ margin_out, const float* __restrict__ mu = nullptr) {
    int warp = (int)(((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    int total = tiles * n;
    if (warp >= total) return;
    int t = warp / n, i = warp - t * n;
    const float* up = Lam0 + ((size_t)t * rows_pad + i) * wp0;
    const float* lo = Lam0 + ((size_t)t * rows_pad + n + i) * wp0;
    const float* sg = sigma + (size_t)t * wp0;
    float su = 0.f, sl = 0.f, du = 0.f, dl = 0.f;        // du, dl: (Lam_0 - J) mu   (non-centred boxes)
    float au = 0.f, al = 0.f;                            // sums of |(Lam_0 - J) mu|: what the rounding of du, dl scales with
    const float* mt = mu ? mu + (size_t)t * wp0 : nullptr;
    if (Jgiven) {
        const float* Jr = Jgiven + ((size_t)t * n + i) * N;
        for (int j = lane; j < N; j += 32) {
            float jv = Jr[j], s = sg[j];
            su += fabsf(up[j] - jv) * s;
            sl += fabsf(lo[j] - jv) * s;
            if (mt) {
                const float pa = (up[j] - jv) * mt[j], pb = (lo[j] - jv) * mt[j];
                du += pa; dl += pb; au += fabsf(pa); al += fabsf(pb);
            }
        }
    } else {
        const float* Jr = Lam0 + ((size_t)t * rows_pad + 2 * n + i) * wp0;
        for (int j = lane * 4; j < wp0; j += 128) {
            float4 a = *reinterpret_cast<const float4*>(up + j), b = *reinterpret_cast<const float4*>(lo + j);
            float4 c = *reinterpret_cast<const float4*>(Jr + j), s = *reinterpret_cast<const float4*>(sg + j);
            su += fabsf(a.x - c.x) * s.x + fabsf(a.y - c.y) * s.y + fabsf(a.z - c.z) * s.z + fabsf(a.w - c.w) * s.w;
            sl += fabsf(b.x - c.x) * s.x + fabsf(b.y - c.y) * s.y + fabsf(b.z - c.z) * s.z + fabsf(b.w - c.w) * s.w;
            if (mt) {
                float4 m = *reinterpret_cast<const float4*>(mt + j);
                const float pa[4] = {(a.x - c.x) * m.x, (a.y - c.y) * m.y, (a.z - c.z) * m.z, (a.w - c.w) * m.w};
                const float pb[4] = {(b.x - c.x) * m.x, (b.y - c.y) * m.y, (b.z - c.z) * m.z, (b.w - c.w) * m.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) { du += pa[q]; dl += pb[q]; au += fabsf(pa[q]); al += fabsf(pb[q]); }
            }
        }
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) {
        su += __shfl_xor_sync(0xffffffffu, su, off); sl += __shfl_xor_sync(0xffffffffu, sl, off);
        du += __shfl_xor_sync(0xffffffffu, du, off); dl += __shfl_xor_sync(0xffffffffu, dl, off);
        au += __shfl_xor_sync(0xffffffffu, au, off); al += __shfl_xor_sync(0xffffffffu, al, off);
    }
    if (lane == 0) {
        float hi = (su + du) + gap[(size_t)t * rows_pad + i];
        float lo_v = (dl - sl) + gap[(size_t)t * rows_pad + n + i];
        float mg = 0.f;
        if (cert) {
            // certified mode: outward-rounded terms (the gap sums carry the chain steps' pads) + eta (the exact nominal
            // output against the centre the chain was developed around); margin_out = eta, the rounding of these sums and
            // the chain pads inside the gap sum (marg, gathered by row_margin_kernel when a margin report is asked for)
            const float gu = gap[(size_t)t * rows_pad + i], gl = gap[(size_t)t * rows_pad + n + i], et = eta[(size_t)t * ld_eta + i];
            const float km = __fmul_ru(__fadd_ru(kap_sum, -1.f), 1.0001f);       // relative rounding of the signed sums du, dl against au, al
            const float pu = __fadd_ru(__fadd_ru(__fadd_ru(__fmul_ru(su, kap_sum), __fmul_ru(gu, kap_gap)), et), __fadd_ru(du, __fmul_ru(au, km)));
            const float pl = __fadd_ru(__fadd_ru(__fadd_ru(__fmul_ru(sl, kap_sum), __fmul_ru(-gl, kap_gap)), et), __fadd_ru(-dl, __fmul_ru(al, km)));
            mg = fmaxf(__fadd_ru(pu, -hi), __fadd_ru(pl, lo_v));
            if (margin_out) mg = __fadd_ru(mg, fmaxf(marg[(size_t)t * rows_pad + i], marg[(size_t)t * rows_pad + n + i]));
            hi = pu; lo_v = -pl;
        }
        if (!(fabsf(hi) <= 3.0e38f) || !(fabsf(lo_v) <= 3.0e38f)) {   // NaN / Inf anywhere in the tile's inputs
            hi = INFINITY; lo_v = -INFINITY; mg = INFINITY;
            atomicExch(domain_flag, 1);
        }
        r_hi[(size_t)t * ld_out + i] = hi;
        r_lo[(size_t)t * ld_out + i] = lo_v;
        if (margin_out) margin_out[(size_t)t * ld_out + i] = mg;
    }
}

// ------------------------------------------------------------------------------------------
// VJP kernels
// ------------------------------------------------------------------------------------------
// Seeds of target s: one CTA per tile; thread j owns input column(s) j, loops over the rows.
//   hidden: Lbar0[up k] = ubar_k sign(Lam_up_0) sigma,  Lbar0[lo k] = -lbar_k sign(Lam_lo_0) sigma
//   output: with S = sign(Lam_0 - J): Lbar0[up i] = g_hi_i S_up sigma, Lbar0[lo i] = -g_lo_i S_lo sigma,
//           Lbar0[jac i] = -(Lbar0[up i] + Lbar0[lo i])
//   rad_bar_j += sum_rows |.| weights;  gapbar[up] = ybar_up, gapbar[lo] = ybar_lo
template <bool MU>
__global__ void __launch_bounds__(256) seed_kernel(int is_out, int rows_pad, int rows_kind, int wp0, const float* __restrict__ Lam0,
                            const float* __restrict__ sigma, const float* __restrict__ ybar_up, const float* __restrict__ ybar_lo,
                            int ldy, float* __restrict__ Lbar0, float* __restrict__ gapbar, float* __restrict__ rad_bar,
                            const float* __restrict__ mu = nullptr, float* __restrict__ mu_bar = nullptr) {
    // grid (tiles, ceil(rows_kind / 32)): a block takes 32 bound indices k of one tile.  64 lanes x float4 cover 256 input
    // columns, the four 64-lane groups take every fourth k; the column sums are joined in shared memory in a fixed order.
    __shared__ float4 red_s[3][64], red_m[3][64];
    const int t = blockIdx.x, k0 = blockIdx.y * 32, k1 = min(k0 + 32, rows_kind);
    const float* base = Lam0 + (size_t)t * rows_pad * wp0;
    float* obase = Lbar0 + (size_t)t * rows_pad * wp0;
    for (int k = k0 + threadIdx.x; k < k1; k += blockDim.x) {
        gapbar[(size_t)t * rows_pad + k] = ybar_up[(size_t)t * ldy + k];
        gapbar[(size_t)t * rows_pad + rows_kind + k] = ybar_lo[(size_t)t * ldy + k];
    }
    if (blockIdx.y == 0)
        for (int r = 2 * rows_kind + threadIdx.x; r < rows_pad; r += blockDim.x) gapbar[(size_t)t * rows_pad + r] = 0.f;
    const int rq = threadIdx.x >> 6, lane64 = threadIdx.x & 63;
    auto sgn = [](float v) { return (float)((v > 0.f) - (v < 0.f)); };
    for (int j0 = 0; j0 < wp0; j0 += 256) {
        const int j = j0 + lane64 * 4;
        const bool on = j < wp0;
        float4 s = make_float4(0.f, 0.f, 0.f, 0.f), m = s, sb = s, mb = s;
        if (on) {
            s = *reinterpret_cast<const float4*>(sigma + (size_t)t * wp0 + j);
            if (MU) m = *reinterpret_cast<const float4*>(mu + (size_t)t * wp0 + j);   // non-centred boxes: y = Lam mu +- |Lam| sigma + gap
#pragma unroll 4
            for (int k = k0 + rq; k < k1; k += 4) {
                const float yu = ybar_up[(size_t)t * ldy + k], yl = ybar_lo[(size_t)t * ldy + k];
                float4 a = *reinterpret_cast<const float4*>(base + (size_t)k * wp0 + j);
                float4 b = *reinterpret_cast<const float4*>(base + (size_t)(rows_kind + k) * wp0 + j);
                if (is_out) {
                    const float4 jv = *reinterpret_cast<const float4*>(base + (size_t)(2 * rows_kind + k) * wp0 + j);
                    a.x -= jv.x; a.y -= jv.y; a.z -= jv.z; a.w -= jv.w;
                    b.x -= jv.x; b.y -= jv.y; b.z -= jv.z; b.w -= jv.w;
                }
                const float4 lu = make_float4(yu * (sgn(a.x) * s.x + m.x), yu * (sgn(a.y) * s.y + m.y), yu * (sgn(a.z) * s.z + m.z),
                                              yu * (sgn(a.w) * s.w + m.w));
                const float4 ll = make_float4(yl * (m.x - sgn(b.x) * s.x), yl * (m.y - sgn(b.y) * s.y), yl * (m.z - sgn(b.z) * s.z),
                                              yl * (m.w - sgn(b.w) * s.w));
                *reinterpret_cast<float4*>(obase + (size_t)k * wp0 + j) = lu;
                *reinterpret_cast<float4*>(obase + (size_t)(rows_kind + k) * wp0 + j) = ll;
                if (is_out)
                    *reinterpret_cast<float4*>(obase + (size_t)(2 * rows_kind + k) * wp0 + j) =
                        make_float4(-(lu.x + ll.x), -(lu.y + ll.y), -(lu.z + ll.z), -(lu.w + ll.w));
                sb.x += yu * fabsf(a.x) - yl * fabsf(b.x); sb.y += yu * fabsf(a.y) - yl * fabsf(b.y);
                sb.z += yu * fabsf(a.z) - yl * fabsf(b.z); sb.w += yu * fabsf(a.w) - yl * fabsf(b.w);
                if (MU) {
                    mb.x += yu * a.x + yl * b.x; mb.y += yu * a.y + yl * b.y;
                    mb.z += yu * a.z + yl * b.z; mb.w += yu * a.w + yl * b.w;
                }
            }
        }
        __syncthreads();
        if (rq > 0) { red_s[rq - 1][lane64] = sb; if (MU) red_m[rq - 1][lane64] = mb; }
        __syncthreads();
        if (rq == 0 && on) {
            for (int q = 0; q < 3; ++q) {
                const float4 v = red_s[q][lane64];
                sb.x += v.x; sb.y += v.y; sb.z += v.z; sb.w += v.w;
                if (MU) { const float4 u = red_m[q][lane64]; mb.x += u.x; mb.y += u.y; mb.z += u.z; mb.w += u.w; }
            }
            float* rb = rad_bar + (size_t)t * wp0 + j;
            atomicAdd(rb, sb.x); atomicAdd(rb + 1, sb.y); atomicAdd(rb + 2, sb.z); atomicAdd(rb + 3, sb.w);
            if (MU && mu_bar) {
                float* mp = mu_bar + (size_t)t * wp0 + j;
                atomicAdd(mp, mb.x); atomicAdd(mp + 1, mb.y); atomicAdd(mp + 2, mb.z); atomicAdd(mp + 3, mb.w);
            }
        }
    }
}

// adjoint of the relaxation parameters of layer l -> (lbar, ubar), and the direct zhat terms
__global__ void relax_vjp_kernel(int act, int tiles, int w_valid, int wp, const float* __restrict__ zhat,
                                 const float* __restrict__ lb, const float* __restrict__ ub, const float* __restrict__ kUb,
                                 const float* __restrict__ kLb, const float* __restrict__ gUb, const float* __restrict__ gLb,
                                 const float* __restrict__ dpb, float* __restrict__ lbar, float* __restrict__ ubar,
                                 float* __restrict__ zbar, int is_layer1, const float* __restrict__ alpha = nullptr) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) { lbar[q] = 0.f; ubar[q] = 0.f; continue; }
        double z = zhat[q], l = lb[q], u = ub[q];
        Relax r = relax_any(act, l, u);
        if (alpha && r.cL == LINE_RELU_LOW) r.kL = (double)alpha[q];
        double gu = gUb[q], gl = gLb[q];
        // g = k zhat + b - phi(zhat):  k_bar_eff = k_bar + zhat g_bar,  b_bar = g_bar
        double kbu = (double)kUb[q] + z * gu, kbl = (double)kLb[q] + z * gl;
        double lo = 0.0, up = 0.0;
        line_vjp(act, r.cU, true, l, u, r.dU, kbu, gu, lo, up, r.tl, r.tu);
        line_vjp(act, r.cL, false, l, u, r.dL, kbl, gl, lo, up, r.tl, r.tu);
        double d1 = act_d1(act, z);
        double zb = (r.kU - d1) * gu + (r.kL - d1) * gl + act_d2(act, z) * (double)dpb[q];
        // l_s = zhat_s - ..., u_s = zhat_s + ...: both pass their adjoint straight to zhat_s
        zb += lo + up;
        lbar[q] = (float)lo;
        ubar[q] = (float)up;
        zbar[q] += (float)zb;
        (void)is_layer1;
    }
}

// ------------------------------------------------------------------------------------------
// CROWN-IBP mode (LEB_FLAG_IBP_HIDDEN): hidden layers s = 2..L-1 bounded by interval propagation of the previous layer's
// bounds instead of back-substitution (PAPER.md:L194-196 leaves the CROWN variant open).  In deviation form:
// a_{s-1} - ahat_{s-1} in [dl, du] = [phi(l) - phi(zhat), phi(u) - phi(zhat)] (phi monotone), centre dc, radius dr;
// z_s - zhat_s in W_s dc -+ |W_s| dr.
// ------------------------------------------------------------------------------------------
__global__ void ibp_dev_kernel(int act, int tiles, int w_valid, int wp, const float* __restrict__ zhat, const float* __restrict__ lb,
                               const float* __restrict__ ub, float* __restrict__ dc, float* __restrict__ dr) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) { dc[q] = 0.f; dr[q] = 0.f; continue; }
        const double f = act_f(act, (double)zhat[q]);
        const double dl = act_f(act, (double)lb[q]) - f, du = act_f(act, (double)ub[q]) - f;
        dc[q] = (float)(0.5 * (du + dl));
        dr[q] = (float)(0.5 * (du - dl));
    }
}

// certified CROWN-IBP: rigorous centre / radius of the activation deviation phi(z) - ahat on [l, u] (phi monotone):
// [phi(l) - ahat, phi(u) - ahat] is contained in dc -+ dr with dc, dr as stored (dr rounded up; libm within 1e-15)
__global__ void ibp_dev_cert_kernel(int act, int tiles, int w_valid, int wp, const float* __restrict__ ahat, const float* __restrict__ lb,
                                    const float* __restrict__ ub, float* __restrict__ dc, float* __restrict__ dr, float* __restrict__ da) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) { dc[q] = 0.f; dr[q] = 0.f; da[q] = 0.f; continue; }
        const double a = (double)ahat[q];
        const double lo = act_f(act, (double)lb[q]) - a - 1e-15, hi = act_f(act, (double)ub[q]) - a + 1e-15;
        const float m = (float)(0.5 * (lo + hi));
        dc[q] = m;
        dr[q] = __double2float_ru(fmax(hi - (double)m, (double)m - lo));
        da[q] = fabsf(m);
    }
}
__global__ void ibp_bounds_kernel(int tiles, int w_valid, int wp, const float* __restrict__ zhat, const float* __restrict__ zc,
                                  const float* __restrict__ zr, float* __restrict__ lb, float* __restrict__ ub) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) { lb[q] = 0.f; ub[q] = 0.f; continue; }
        const float z = zhat[q], m = zc[q], r = zr[q];
        lb[q] = z + (m - r);
        ub[q] = z + (m + r);
    }
}

// reverse: seeds of the two products from the (complete) adjoints of (l_s, u_s)
__global__ void ibp_seed_kernel(size_t count, const float* __restrict__ lbar, const float* __restrict__ ubar, float* __restrict__ zcb,
                                float* __restrict__ zrb) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x) {
        const float l = lbar[q], u = ubar[q];
        zcb[q] = l + u;
        zrb[q] = u - l;
    }
}

// reverse: (dc_bar, dr_bar) of layer s-1 -> what layer s's interval step sends to (l_{s-1}, u_{s-1}) and to zhat_{s-1}
__global__ void ibp_bwd_kernel(int act, int tiles, int w_valid, int wp, const float* __restrict__ zhat, const float* __restrict__ lb,
                               const float* __restrict__ ub, const float* __restrict__ dcb, const float* __restrict__ drb,
                               float* __restrict__ ibl, float* __restrict__ ibu, float* __restrict__ zbar) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid) { ibl[q] = 0.f; ibu[q] = 0.f; continue; }
        const double dlb = 0.5 * ((double)dcb[q] - (double)drb[q]), dub = 0.5 * ((double)dcb[q] + (double)drb[q]);
        ibl[q] = (float)(act_d1(act, (double)lb[q]) * dlb);
        ibu[q] = (float)(act_d1(act, (double)ub[q]) * dub);
        zbar[q] += (float)(-act_d1(act, (double)zhat[q]) * (dlb + dub));
    }
}

// reverse: add what the next layer's interval step sent; l = zhat + ..., u = zhat + ... pass it on to zhat as well
__global__ void ibp_add_kernel(size_t count, float* __restrict__ lbar, float* __restrict__ ubar, float* __restrict__ zbar,
                               const float* __restrict__ ibl, const float* __restrict__ ibu) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x) {
        const float a = ibl[q], b = ibu[q];
        lbar[q] += a;
        ubar[q] += b;
        zbar[q] += a + b;
    }
}

// ub1 - lb1 adjoint for the layer-1 radius |W_1| sigma
__global__ void diff_kernel(const float* __restrict__ ubar, const float* __restrict__ lbar, float* __restrict__ out, size_t count) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x)
        out[q] = ubar[q] - lbar[q];
}

// alpha-CROWN style refinement: one projected gradient step on the lower slopes of the unstable ReLU neurons;
// d(objective)/d(alpha) = k_bar^L + zhat gap_bar^L (gap^L = alpha zhat - relu(zhat))
// keep the slopes of the tiles whose last iterate was the tightest so far
__global__ void alpha_keep_kernel(int tiles, int wp, const int* __restrict__ take, const float* __restrict__ alpha, float* __restrict__ best) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x)
        if (take[q / wp]) best[q] = alpha[q];
}
__global__ void alpha_update_kernel(int tiles, int w_valid, int wp, const float* __restrict__ zhat, const float* __restrict__ lb,
                                    const float* __restrict__ ub, const float* __restrict__ kLb, const float* __restrict__ gLb,
                                    float* __restrict__ alpha, float lr) {
    size_t total = (size_t)tiles * wp;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % wp);
        if (c >= w_valid || !(lb[q] < 0.f && ub[q] > 0.f)) continue;
        const float g = kLb[q] + zhat[q] * gLb[q];
        const float a = alpha[q] - lr * g;
        if (a == a) alpha[q] = fminf(fmaxf(a, 0.f), 1.f);
    }
}

// keep the tightest iterate of every tile: one block per tile
// first: 1 = the adaptive-slope iterate (sets width0), 0 = a later iterate (taken if tighter), 2 = the final evaluation at the kept
// slopes (always taken; width0 untouched)
__global__ void alpha_best_kernel(int n, int ld_out, int first, const float* __restrict__ cur_lo, const float* __restrict__ cur_hi,
                                  float* __restrict__ r_lo, float* __restrict__ r_hi, float* __restrict__ w0, float* __restrict__ wbest,
                                  int* __restrict__ take_out) {
    __shared__ float red[8];
    __shared__ int take;
    const size_t t = blockIdx.x;
    float w = 0.f;
    for (int i = threadIdx.x; i < n; i += blockDim.x) w += cur_hi[t * n + i] - cur_lo[t * n + i];
    for (int off = 16; off; off >>= 1) w += __shfl_xor_sync(0xffffffffu, w, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = w;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) tot += red[q];
        if (first == 1) { w0[t] = tot; wbest[t] = tot; take = 1; }
        else if (first == 2 || tot < wbest[t]) { wbest[t] = tot; take = 1; }
        else take = 0;
        take_out[t] = take;
    }
    __syncthreads();
    if (take)
        for (int i = threadIdx.x; i < n; i += blockDim.x) { r_lo[t * ld_out + i] = cur_lo[t * n + i]; r_hi[t * ld_out + i] = cur_hi[t * n + i]; }
}

__global__ void abs_kernel(const float* __restrict__ a, float* __restrict__ out, size_t count) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x) out[q] = fabsf(a[q]);
}

__global__ void sum_kernel(const float* __restrict__ a, const float* __restrict__ b, float* __restrict__ out, size_t count) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += (size_t)gridDim.x * blockDim.x)
        out[q] = a[q] + b[q];
}

__global__ void write_grads_kernel(int tiles, int N, int wp0, int ld_in, const float* __restrict__ nom_bar,
                                   const float* __restrict__ rad_bar, float* __restrict__ grad_nom, float* __restrict__ grad_rad,
                                   const float* __restrict__ mu_bar = nullptr, float* __restrict__ grad_mu = nullptr) {
    size_t total = (size_t)tiles * N;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(q / N), c = (int)(q - (size_t)t * N);
        grad_nom[(size_t)t * ld_in + c] = nom_bar[(size_t)t * wp0 + c];
        grad_rad[(size_t)t * ld_in + c] = rad_bar[(size_t)t * wp0 + c];
        if (grad_mu) grad_mu[(size_t)t * ld_in + c] = mu_bar[(size_t)t * wp0 + c];
    }
}

__global__ void copy_hidden_kernel(int tiles, int w, int wp, const float* __restrict__ lb, const float* __restrict__ ub,
                                   float* __restrict__ l, float* __restrict__ u) {
    size_t total = (size_t)tiles * w;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int t = (int)(q / w), c = (int)(q - (size_t)t * w);
        l[q] = lb[(size_t)t * wp + c];
        u[q] = ub[(size_t)t * wp + c];
    }
}

// Lambda_0 rows of one target: [tiles x rows_pad x wp0] (upper | lower | ...) -> [tiles x 2 x rows x N]
__global__ void copy_coeffs_kernel(int tiles, int rows, int rows_kind, int rows_pad, int N, int wp0, const float* __restrict__ Lam0,
                                   float* __restrict__ out) {
    size_t total = (size_t)tiles * 2 * rows * N;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % N);
        size_t r = q / N;
        int k = (int)(r % rows), chain = (int)((r / rows) % 2), t = (int)(r / ((size_t)2 * rows));
        out[q] = Lam0[((size_t)t * rows_pad + (size_t)chain * rows_kind + k) * wp0 + c];
    }
}

inline unsigned gs_grid(size_t work) {
    size_t b = (work + 255) / 256;
    if (b > 148 * 16) b = 148 * 16;
    if (b < 1) b = 1;
    return (unsigned)b;
}

// ------------------------------------------------------------------------------------------
// GEMM launch helpers
// ------------------------------------------------------------------------------------------
// kc / flops: kernel class and algorithmic flops (true, unpadded dims) for the profiling aid
template <int AMODE, int EPI>
void launch_gemm(NnState* S, const GemmArgs& g, cudaStream_t st, long long* launches, int kc = LEB_KC_NN_OTHER, double flops = 0.0) {
    dim3 grid((g.N + BN - 1) / BN, (g.M + BM - 1) / BM);
    S->prof->begin(kc, st);
    gemm_ffma_kernel<AMODE, EPI><<<grid, GT, 0, st>>>(g);
    S->prof->end(kc, st, flops);
    ++*launches;
}

GemmArgs plain_args(int M, int N, int K, const float* A, int lda, const float* B, int ldb, float* C, int ldc) {
    GemmArgs g{};
    g.M = M; g.N = N; g.K = K; g.A = A; g.lda = lda; g.B = B; g.ldb = ldb; g.C = C; g.ldc = ldc;
    g.rows_pad = 1; g.rows_kind = 1; g.nkinds = 1;
    return g;
}

void* ws_alloc(NnState* S, size_t bytes, bool* ok) {
    void* p = nullptr;
    if (bytes == 0) bytes = 16;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { *ok = false; return nullptr; }
    S->allocs.push_back(p);
    return p;
}

void ws_free(NnState* S) {
    for (void* p : S->allocs) cudaFree(p);
    S->allocs.clear();
    S->chunk = 0;
    S->ws_vjp = false;
    S->last_tiles = 0;
}

size_t bytes_per_tile(const NnState* S, bool vjp) {
    size_t f = 5 * (size_t)S->wp[0] + (size_t)S->wp[1];
    for (int l = 1; l < S->L; ++l) f += (size_t)S->wp[l] * (vjp ? 24 : 16);
    size_t maxLam = 0;
    for (int s = 2; s <= S->L; ++s) {
        for (int l = 0; l <= s - 2; ++l) f += (size_t)S->rows_pad[s] * S->wp[l];
        f += (size_t)S->rows_pad[s] + (s == S->L ? S->rows_pad[s] : 0);
        for (int l = 0; l <= s - 2; ++l) maxLam = std::max(maxLam, (size_t)S->rows_pad[s] * S->wp[l]);
    }
    if (vjp) f += 2 * maxLam + 2 * (size_t)S->wp[0] + 2 * (size_t)S->w[S->L] + 1024;
    return f * sizeof(float);
}

// (re)allocate the chunk workspace
leb_status ensure_workspace(NnState* S, int tiles, bool vjp) {
    // Default: the whole batch resident (config 5: 6 400 tiles x 17 MB = 108 GB of the 180 GB HBM) -- one launch per chain
    // step, and leb_vjp can reuse the forward's coefficient blocks (LEB_FLAG_REUSE_FWD) -- capped by 85 % of the free
    // memory.  The workspace is always sized for the reverse sweep too, so that a later leb_vjp does not reallocate.
    (void)vjp;
    int want = S->chunk_req > 0 ? S->chunk_req : tiles;
    if (want > tiles && tiles > 0) want = tiles;
    if (S->chunk >= want || (S->chunk > 0 && S->chunk_capped && S->chunk_req == 0)) return LEB_OK;
    cudaDeviceSynchronize();
    ws_free(S);
    S->chunk_capped = false;
    {
        size_t free_b = 0, total_b = 0;
        const size_t per = bytes_per_tile(S, true);
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && per > 0) {
            const size_t fit = (size_t)(0.85 * (double)free_b) / per;
            if ((size_t)want > fit) { want = fit < 1 ? 1 : (int)fit; S->chunk_capped = true; }
        }
        int maxrows = 1;                                   // the FFMA kernels put M / 128 row blocks on grid.y (<= 65535)
        for (int s = 2; s <= S->L; ++s) maxrows = std::max(maxrows, S->rows_pad[s]);
        const int lim = (int)((size_t)65535 * 128 / (size_t)maxrows);
        if (want > lim) { want = lim; S->chunk_capped = true; }
    }
    vjp = true;
    const int C = want, L = S->L;
    bool ok = true;
    auto F = [&](size_t count) { return (float*)ws_alloc(S, count * sizeof(float), &ok); };
    S->nomp = F((size_t)C * S->wp[0]);
    S->radp = F((size_t)C * S->wp[0]);
    S->rad1 = F((size_t)C * S->wp[1]);
    S->mup = F((size_t)C * S->wp[0]);
    S->mu1 = F((size_t)C * S->wp[1]);
    S->mu_bar = F((size_t)C * S->wp[0]);
    S->alpha_take = (int*)F((size_t)C);
    {
        int mw = 0;
        for (int l = 1; l < L; ++l) mw = std::max(mw, S->wp[l]);
        for (float** p : {&S->ibp_c, &S->ibp_r, &S->ibp_a, &S->ibp_m, &S->ibp_vm}) *p = F((size_t)C * mw);
    }
    for (int l = 1; l < L; ++l) {
        size_t c = (size_t)C * S->wp[l];
        S->zhat[l] = F(c); S->ahat[l] = F(c); S->dphi[l] = F(c); S->lb[l] = F(c); S->ub[l] = F(c);
        S->kU[l] = F(c); S->kL[l] = F(c); S->gU[l] = F(c); S->gL[l] = F(c);
        S->ce[l] = F(c); S->ct[l] = F(c); S->cv[l] = F(c); S->adev[l] = F(c); S->mU[l] = F(c); S->mL[l] = F(c);
        S->alpha[l] = F(c); S->alpha_best[l] = F(c);
        if (vjp) {
            S->kUb[l] = F(c); S->kLb[l] = F(c); S->gUb[l] = F(c); S->gLb[l] = F(c); S->dpb[l] = F(c);
            S->zbar[l] = F(c); S->lbar[l] = F(c); S->ubar[l] = F(c);
        }
    }
    size_t maxLam = 0;
    for (int s = 2; s <= L; ++s) {
        for (int l = 0; l <= s - 2; ++l) {
            size_t c = (size_t)C * S->rows_pad[s] * S->wp[l];
            S->Lam[s][l] = F(c);
            maxLam = std::max(maxLam, c);
        }
        S->gap[s] = F((size_t)C * S->rows_pad[s]);
    }
    S->marg = F((size_t)C * S->rows_pad[L]);
    S->eta = F((size_t)C * S->wp[L]);
    if (vjp) {
        S->Lbar[0] = F(maxLam);
        S->Lbar[1] = F(maxLam);
        size_t maxrows = 0;
        for (int s = 2; s <= L; ++s) maxrows = std::max(maxrows, (size_t)S->rows_pad[s]);
        S->gapbar = F((size_t)C * maxrows);
        S->nom_bar = F((size_t)C * S->wp[0]);
        S->rad_bar = F((size_t)C * S->wp[0]);
        S->glo_p = F((size_t)C * S->w[L]);
        S->ghi_p = F((size_t)C * S->w[L]);
    }
    if (!ok) { ws_free(S); return LEB_ERR_NOMEM; }
    S->chunk = C;
    S->ws_vjp = vjp;
    return LEB_OK;
}

// forward for one chunk of C tiles whose padded inputs are already in S->nomp / S->radp
void launch_cert_layer(NnState* S, int C, int l, bool out_only, cudaStream_t st, long long* launches) {
    const int J = out_only ? S->w[l] : S->wp[l], K = S->wp[l - 1];
    dim3 grid((J + CJ - 1) / CJ, (C + CM - 1) / CM);
    const float* X = (l == 1) ? S->nomp : S->ahat[l - 1];
    const float* T = (l == 1) ? nullptr : S->ct[l - 1];
    const float* A = (l == 1) ? S->radp : S->adev[l - 1];
    if (out_only)
        cert_layer_kernel<<<grid, 256, 0, st>>>(C, J, K, S->Wt[l], S->rowsW[l], S->bias[l], nullptr, T, nullptr, K, nullptr, nullptr, S->act, 1,
                                               nullptr, S->eta, nullptr, S->wp[l]);
    else
        cert_layer_kernel<<<grid, 256, 0, st>>>(C, J, K, S->Wt[l], S->rowsW[l], S->bias[l], X, T, A, K, S->zhat[l], S->ahat[l], S->act, 0,
                                               S->ce[l], S->ct[l], S->cv[l], S->wp[l]);
    ++*launches;
}

void forward_chunk(NnState* S, int C, const float* Jgiven, bool with_jac, bool cert, bool marg_report, cudaStream_t st,
                   long long* launches, bool ibp = false) {
    const int L = S->L;
    int ksum = 0;                                   // total contraction length of the gap sums of the deepest chain
    for (int l = 1; l < L; ++l) ksum += S->wp[l];
    const float kap_sum = 1.f + (float)(S->wp[0] + 8) * 1.1920929e-07f, kap_gap = 1.f + (float)(ksum + 64) * 1.1920929e-07f;
    // ---- N1 nominal pass
    const float* a_prev = S->nomp;
    for (int l = 1; l < L; ++l) {
        GemmArgs g = plain_args(C, S->wp[l], S->wp[l - 1], a_prev, S->wp[l - 1], S->Wt[l], S->wp[l], S->zhat[l], S->wp[l]);
        g.bias = S->bias[l]; g.ahat = S->ahat[l]; g.dphi_out = S->dphi[l]; g.act = S->act;
        launch_gemm<AMODE_PLAIN, EPI_NOMINAL>(S, g, st, launches);
        a_prev = S->ahat[l];
    }
    // ---- N2 layer-1 interval bounds: rad1 = |W_1| sigma
    if (cert) {
        // certified: the radius is the rounded-up product v_1 = |W_1| sigma, widened by the centre residual e_1
        launch_cert_layer(S, C, 1, false, st, launches);
        const float* m1 = nullptr;
        const float* vmu = nullptr;
        if (S->mu_cur) {
            // non-centred boxes: mu1 = W_1 mu (FP32 product, nearest) and its rounding scale rad1 = |W_1||mu| (rounded up; the
            // value-mode radius array is free in certified mode; the cert kernel's e / t outputs of this call go to scratch)
            GemmArgs gm = plain_args(C, S->wp[1], S->wp[0], S->mu_cur, S->wp[0], S->Wt[1], S->wp[1], S->mu1, S->wp[1]);
            launch_gemm<AMODE_PLAIN, EPI_STORE>(S, gm, st, launches);
            abs_kernel<<<gs_grid((size_t)C * S->wp[0]), 256, 0, st>>>(S->mu_cur, S->mu_bar, (size_t)C * S->wp[0]);
            dim3 grid((S->wp[1] + CJ - 1) / CJ, (C + CM - 1) / CM);
            cert_layer_kernel<<<grid, 256, 0, st>>>(C, S->wp[1], S->wp[0], S->Wt[1], S->rowsW[1], S->bias[1], S->nomp, nullptr, S->mu_bar, S->wp[0],
                                                   S->zhat[1], S->ahat[1], S->act, 0, S->mU[1], S->mL[1], S->rad1, S->wp[1]);
            *launches += 2;
            m1 = S->mu1; vmu = S->rad1;
        }
        relax_fwd_cert_kernel<<<gs_grid((size_t)C * S->wp[1]), 256, 0, st>>>(
            S->act, C, S->w[1], S->wp[1], 1, S->use_tc ? 1 : 0, S->zhat[1], S->ahat[1], S->cv[1], S->ce[1], S->lb[1], S->ub[1], S->kU[1],
            S->kL[1], S->gU[1], S->gL[1], S->adev[1], S->mU[1], S->mL[1], m1, vmu, (float)(S->wp[0] + 4) * 5.9604652e-08f * 1.000001f,
            S->alpha_mode == 2 ? S->alpha[1] : nullptr);
        ++*launches;
    } else {
        GemmArgs g = plain_args(C, S->wp[1], S->wp[0], S->radp, S->wp[0], S->Wabs1t, S->wp[1], S->rad1, S->wp[1]);
        launch_gemm<AMODE_PLAIN, EPI_STORE>(S, g, st, launches);
        if (S->mu_cur) {      // non-centred boxes: the centre of z_1 - zhat_1 is W_1 mu
            GemmArgs gm = plain_args(C, S->wp[1], S->wp[0], S->mu_cur, S->wp[0], S->Wt[1], S->wp[1], S->mu1, S->wp[1]);
            launch_gemm<AMODE_PLAIN, EPI_STORE>(S, gm, st, launches);
        }
        relax_fwd_kernel<<<gs_grid((size_t)C * S->wp[1]), 256, 0, st>>>(S->act, C, S->w[1], S->wp[1], S->zhat[1], S->rad1, S->lb[1],
                                                                      S->ub[1], S->kU[1], S->kL[1], S->gU[1], S->gL[1],
                                                                      S->mu_cur ? S->mu1 : nullptr, S->alpha[1], S->alpha_mode);
        ++*launches;
    }
    // ---- N3 / N4: targets s = 2 .. L
    for (int s = 2; s <= L; ++s) {
        const bool is_out = (s == L);
        const int nk = is_out ? (with_jac ? 3 : 2) : 2;
        const int rp = S->rows_pad[s], rk = S->rows_kind[s];
        if (ibp && !is_out && cert) {
            // certified CROWN-IBP: z_s - c_s = W_s (a_{s-1} - ahat_{s-1}) + (centre residual), a_{s-1} - ahat_{s-1} in dc -+ dr, so
            // z_s - c_s in m -+ (|W_s| dr + gam |W_s||dc| + e_s), m = the FP32 product W_s dc (wrong by at most gam |W_s||dc|): the
            // layer-1 formula of a non-centred box with (mu, sigma) -> (dc, dr), every |W| product rounded up (cert_layer_kernel)
            const size_t cp = (size_t)C * S->wp[s - 1], cs = (size_t)C * S->wp[s];
            launch_cert_layer(S, C, s, false, st, launches);                    // e_s, t_s
            ibp_dev_cert_kernel<<<gs_grid(cp), 256, 0, st>>>(S->act, C, S->w[s - 1], S->wp[s - 1], S->ahat[s - 1], S->lb[s - 1], S->ub[s - 1],
                                                            S->ibp_c, S->ibp_r, S->ibp_a);
            GemmArgs gm = plain_args(C, S->wp[s], S->wp[s - 1], S->ibp_c, S->wp[s - 1], S->Wt[s], S->wp[s], S->ibp_m, S->wp[s]);
            launch_gemm<AMODE_PLAIN, EPI_STORE>(S, gm, st, launches);
            dim3 grid((S->wp[s] + CJ - 1) / CJ, (C + CM - 1) / CM);
            cert_layer_kernel<<<grid, 256, 0, st>>>(C, S->wp[s], S->wp[s - 1], S->Wt[s], S->rowsW[s], S->bias[s], S->ahat[s - 1], nullptr, S->ibp_r,
                                                   S->wp[s - 1], S->zhat[s], S->ahat[s], S->act, 0, S->mU[s], S->mL[s], S->cv[s], S->wp[s]);
            cert_layer_kernel<<<grid, 256, 0, st>>>(C, S->wp[s], S->wp[s - 1], S->Wt[s], S->rowsW[s], S->bias[s], S->ahat[s - 1], nullptr, S->ibp_a,
                                                   S->wp[s - 1], S->zhat[s], S->ahat[s], S->act, 0, S->mU[s], S->mL[s], S->ibp_vm, S->wp[s]);
            relax_fwd_cert_kernel<<<gs_grid(cs), 256, 0, st>>>(
                S->act, C, S->w[s], S->wp[s], 1, S->use_tc ? 1 : 0, S->zhat[s], S->ahat[s], S->cv[s], S->ce[s], S->lb[s], S->ub[s], S->kU[s],
                S->kL[s], S->gU[s], S->gL[s], S->adev[s], S->mU[s], S->mL[s], S->ibp_m, S->ibp_vm,
                (float)(S->wp[s - 1] + 4) * 5.9604652e-08f * 1.000001f, S->alpha_mode == 2 ? S->alpha[s] : nullptr);
            *launches += 4;
            continue;
        }
        if (ibp && !is_out) {
            // CROWN-IBP: l_s, u_s = zhat_s + W_s dc -+ |W_s| dr (the cert-mode arrays serve as scratch: value mode only)
            const size_t cp = (size_t)C * S->wp[s - 1], cs = (size_t)C * S->wp[s];
            ibp_dev_kernel<<<gs_grid(cp), 256, 0, st>>>(S->act, C, S->w[s - 1], S->wp[s - 1], S->zhat[s - 1], S->lb[s - 1], S->ub[s - 1],
                                                       S->ce[s - 1], S->ct[s - 1]);
            ++*launches;
            GemmArgs g1 = plain_args(C, S->wp[s], S->wp[s - 1], S->ce[s - 1], S->wp[s - 1], S->Wt[s], S->wp[s], S->cv[s], S->wp[s]);
            launch_gemm<AMODE_PLAIN, EPI_STORE>(S, g1, st, launches);
            GemmArgs g2 = plain_args(C, S->wp[s], S->wp[s - 1], S->ct[s - 1], S->wp[s - 1], S->Wabst[s], S->wp[s], S->adev[s], S->wp[s]);
            launch_gemm<AMODE_PLAIN, EPI_STORE>(S, g2, st, launches);
            ibp_bounds_kernel<<<gs_grid(cs), 256, 0, st>>>(C, S->w[s], S->wp[s], S->zhat[s], S->cv[s], S->adev[s], S->lb[s], S->ub[s]);
            relax_fwd_kernel<<<gs_grid(cs), 256, 0, st>>>(S->act, C, S->w[s], S->wp[s], S->zhat[s], nullptr, S->lb[s], S->ub[s], S->kU[s],
                                                         S->kL[s], S->gU[s], S->gL[s], nullptr, S->alpha[s], S->alpha_mode);
            *launches += 2;
            continue;
        }
        if (cert) launch_cert_layer(S, C, s, is_out, st, launches);     // e_s, t_s, v_s (eta for the output) -- needs adev_{s-1}
        for (int l = s - 1; l >= 1; --l) {
            GemmArgs g{};
            g.M = C * rp; g.N = S->wp[l - 1]; g.K = S->wp[l];
            g.a_shared = (l == s - 1);
            g.A = g.a_shared ? S->W[s] : S->Lam[s][l];
            g.lda = S->wp[l];
            g.B = S->W[l]; g.ldb = S->wp[l - 1];
            g.C = S->Lam[s][l - 1]; g.ldc = S->wp[l - 1];
            g.rows_pad = rp; g.rows_kind = rk; g.nkinds = nk;
            g.kU = S->kU[l]; g.kL = S->kL[l]; g.gU = S->gU[l]; g.gL = S->gL[l]; g.dphi = S->dphi[l]; g.ldp = S->wp[l];
            g.gap = S->gap[s]; g.gap_init = (l == s - 1);
            if (cert && is_out && marg_report) {
                const size_t warps = (size_t)C * 2 * rk;
                row_margin_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>(C, rp, rk, S->wp[l], g.A, g.a_shared, S->mU[l], S->mL[l],
                                                                                     S->marg, l == s - 1);
                ++*launches;
            }
            const double flops = 2.0 * C * nk * (is_out ? S->w[L] : S->w[s]) * (double)S->w[l] * S->w[l - 1];
            if (S->use_tc) {
                S->prof->begin(LEB_KC_CHAIN_FWD, st);
                const cudaError_t le = S->use_pairs ? tc2::launch_chain_gemm_tc2_fwd(g, S->mapWt_hi[l], S->mapWt_lo[l], S->num_sms, st)
                                                    : tc::launch_chain_gemm_tc<tc::MODE_FWD>(g, S->mapWt_hi[l], S->mapWt_lo[l], S->num_sms, st);
                if (le != cudaSuccess) S->launch_failed = true;
                S->prof->end(LEB_KC_CHAIN_FWD, st, flops);
                ++*launches;
            } else {
                launch_gemm<AMODE_CHAIN, EPI_STORE>(S, g, st, launches, LEB_KC_CHAIN_FWD, flops);
            }
        }
        if (!is_out) {
            size_t warps = (size_t)C * rk;
            concretise_hidden_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>(
                C, rp, rk, S->wp[0], S->Lam[s][0], S->radp, S->gap[s], S->zhat[s], S->lb[s], S->ub[s], cert ? S->ce[s] : nullptr,
                kap_sum, kap_gap, S->mu_cur);
            ++*launches;
            if (cert) {
                relax_fwd_cert_kernel<<<gs_grid((size_t)C * S->wp[s]), 256, 0, st>>>(
                    S->act, C, S->w[s], S->wp[s], 0, S->use_tc ? 1 : 0, S->zhat[s], S->ahat[s], S->cv[s], S->ce[s], S->lb[s], S->ub[s],
                    S->kU[s], S->kL[s], S->gU[s], S->gL[s], S->adev[s], S->mU[s], S->mL[s], nullptr, nullptr, 0.f,
                    S->alpha_mode == 2 ? S->alpha[s] : nullptr);
            } else {
                relax_fwd_kernel<<<gs_grid((size_t)C * S->wp[s]), 256, 0, st>>>(S->act, C, S->w[s], S->wp[s], S->zhat[s], nullptr, S->lb[s],
                                                                              S->ub[s], S->kU[s], S->kL[s], S->gU[s], S->gL[s], nullptr,
                                                                              S->alpha[s], S->alpha_mode);
            }
            ++*launches;
        }
    }
    (void)Jgiven;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// state management
// ------------------------------------------------------------------------------------------
NnState* leb_nn_create() { return new NnState(); }

static void free_weights(NnState* S) {
    for (int l = 0; l <= kMaxLayers; ++l) {
        if (S->W[l]) cudaFree(S->W[l]);
        if (S->Wt[l]) cudaFree(S->Wt[l]);
        if (S->bias[l]) cudaFree(S->bias[l]);
        S->W[l] = S->Wt[l] = S->bias[l] = nullptr;
        for (float** p : {&S->Whi[l], &S->Wlo[l], &S->Wthi[l], &S->Wtlo[l], &S->Wabs[l], &S->Wabst[l]}) { if (*p) cudaFree(*p); *p = nullptr; }
    }
    S->tc_ready = false;
    if (S->Wabs1) cudaFree(S->Wabs1);
    if (S->Wabs1t) cudaFree(S->Wabs1t);
    S->Wabs1 = S->Wabs1t = nullptr;
    S->ready = false;
}

void leb_nn_destroy(NnState* S) {
    if (!S) return;
    cudaDeviceSynchronize();
    ws_free(S);
    free_weights(S);
    for (void* p : S->alpha_scratch) cudaFree(p);
    delete S;
}

bool leb_nn_ready(const NnState* S) { return S && S->ready; }
int leb_nn_n(const NnState* S) { return S->w[S->L]; }
int leb_nn_N(const NnState* S) { return S->w[0]; }

leb_status leb_nn_set_chunk(NnState* S, int tiles) {
    if (tiles < 0) return LEB_ERR_ARG;
    S->chunk_req = tiles;
    cudaDeviceSynchronize();
    ws_free(S);
    return LEB_OK;
}

leb_status leb_nn_set_mlp(NnState* S, const leb_mlp* m, cudaStream_t st, long long* launches) {
    if (!m || !m->dims || !m->W || !m->b) return LEB_ERR_ARG;
    if (m->n_layers < 2 || m->n_layers > kMaxLayers) return LEB_ERR_SHAPE;
    if (m->act != LEB_ACT_RELU && m->act != LEB_ACT_TANH) return LEB_ERR_ARG;
    for (int l = 0; l <= m->n_layers; ++l) if (m->dims[l] < 1) return LEB_ERR_SHAPE;
    cudaDeviceSynchronize();
    ws_free(S);
    free_weights(S);
    S->L = m->n_layers;
    S->act = m->act;
    const int L = S->L;
    for (int l = 0; l <= L; ++l) { S->w[l] = m->dims[l]; S->wp[l] = rup(m->dims[l], kPad); }
    bool ok = true;
    std::vector<void*> staged;
    for (int l = 1; l <= L; ++l) {
        const int rows = S->w[l], cols = S->w[l - 1];
        const int rows_p = (l < L) ? S->wp[l] : rows;      // output rows are not padded (they are only A rows)
        const int cols_p = S->wp[l - 1];
        S->rowsW[l] = rows_p;
        const float* src = m->W[l - 1];
        const float* bsrc = m->b[l - 1];
        float *dW = nullptr, *db = nullptr;
        if (m->weights_on_host) {
            ok = ok && cudaMalloc(&dW, (size_t)rows * cols * sizeof(float)) == cudaSuccess;
            ok = ok && cudaMalloc(&db, (size_t)rows * sizeof(float)) == cudaSuccess;
            if (!ok) break;
            staged.push_back(dW); staged.push_back(db);
            cudaMemcpyAsync(dW, src, (size_t)rows * cols * sizeof(float), cudaMemcpyHostToDevice, st);
            cudaMemcpyAsync(db, bsrc, (size_t)rows * sizeof(float), cudaMemcpyHostToDevice, st);
            src = dW; bsrc = db;
        }
        ok = ok && cudaMalloc(&S->W[l], (size_t)rows_p * cols_p * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMalloc(&S->Wt[l], (size_t)rows_p * cols_p * sizeof(float)) == cudaSuccess;
        ok = ok && cudaMalloc(&S->bias[l], (size_t)rup(rows_p, kPad) * sizeof(float)) == cudaSuccess;
        if (!ok) break;
        size_t tot = (size_t)rows_p * cols_p;
        pack_matrix_kernel<<<gs_grid(tot), 256, 0, st>>>(src, rows, cols, cols, S->W[l], rows_p, cols_p, 0, 0);
        pack_matrix_kernel<<<gs_grid(tot), 256, 0, st>>>(src, rows, cols, cols, S->Wt[l], rows_p, cols_p, 1, 0);
        pack_matrix_kernel<<<gs_grid(rows_p), 256, 0, st>>>(bsrc, 1, rows, rows, S->bias[l], 1, rup(rows_p, kPad), 0, 0);
        *launches += 3;
        if (l < L) {
            for (float** p : {&S->Whi[l], &S->Wlo[l], &S->Wthi[l], &S->Wtlo[l]}) ok = ok && cudaMalloc(p, tot * sizeof(float)) == cudaSuccess;
            if (!ok) break;
            split_tf32_kernel<<<gs_grid(tot), 256, 0, st>>>(S->W[l], S->Whi[l], S->Wlo[l], tot);
            split_tf32_kernel<<<gs_grid(tot), 256, 0, st>>>(S->Wt[l], S->Wthi[l], S->Wtlo[l], tot);
            *launches += 2;
        }
        if (l >= 2 && l < L) {
            ok = ok && cudaMalloc(&S->Wabs[l], tot * sizeof(float)) == cudaSuccess;
            ok = ok && cudaMalloc(&S->Wabst[l], tot * sizeof(float)) == cudaSuccess;
            if (!ok) break;
            pack_matrix_kernel<<<gs_grid(tot), 256, 0, st>>>(src, rows, cols, cols, S->Wabs[l], rows_p, cols_p, 0, 1);
            pack_matrix_kernel<<<gs_grid(tot), 256, 0, st>>>(src, rows, cols, cols, S->Wabst[l], rows_p, cols_p, 1, 1);
            *launches += 2;
        }
        if (l == 1) {
            ok = ok && cudaMalloc(&S->Wabs1, tot * sizeof(float)) == cudaSuccess;
            ok = ok && cudaMalloc(&S->Wabs1t, tot * sizeof(float)) == cudaSuccess;
            if (!ok) break;
            pack_matrix_kernel<<<gs_grid(tot), 256, 0, st>>>(src, rows, cols, cols, S->Wabs1, rows_p, cols_p, 0, 1);
            pack_matrix_kernel<<<gs_grid(tot), 256, 0, st>>>(src, rows, cols, cols, S->Wabs1t, rows_p, cols_p, 1, 1);
            *launches += 2;
        }
    }
    cudaStreamSynchronize(st);
    for (void* p : staged) cudaFree(p);
    if (!ok || cudaGetLastError() != cudaSuccess) { free_weights(S); return ok ? LEB_ERR_CUDA : LEB_ERR_NOMEM; }
    for (int s = 2; s <= L; ++s) {
        S->rows_kind[s] = (s < L) ? S->wp[s] : S->w[L];
        S->rows_pad[s] = rup((s < L ? 2 : 3) * S->rows_kind[s], kRowBlock);
    }
    // TMA maps of the split weights (K-major B operands): W[l] is [wp[l] x wp[l-1]], Wt[l] is [wp[l-1] x wp[l]]
    S->tc_ready = true;
    for (int l = 1; l < L; ++l) {
        S->tc_ready = S->tc_ready && tc::make_weight_map(&S->mapW_hi[l], S->Whi[l], S->wp[l], S->wp[l - 1]);
        S->tc_ready = S->tc_ready && tc::make_weight_map(&S->mapW_lo[l], S->Wlo[l], S->wp[l], S->wp[l - 1]);
        S->tc_ready = S->tc_ready && tc::make_weight_map(&S->mapWt_hi[l], S->Wthi[l], S->wp[l - 1], S->wp[l]);
        S->tc_ready = S->tc_ready && tc::make_weight_map(&S->mapWt_lo[l], S->Wtlo[l], S->wp[l - 1], S->wp[l]);
    }
    if (!S->tc_ready) { free_weights(S); return LEB_ERR_CUDA; }   // no silent fallback: the driver must provide cuTensorMapEncodeTiled
    {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&S->num_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    S->ready = true;
    return LEB_OK;
}

// ------------------------------------------------------------------------------------------
// forward
// ------------------------------------------------------------------------------------------
leb_status leb_nn_forward(NnState* S, int tiles, const float* nom, const float* rad, const float* mu, const float* J, int ld_in,
                          float* r_lo, float* r_hi, float* margin, int ld_out, unsigned flags, int* domain_flag, cudaStream_t st,
                          long long* launches, LebProf* prof) {
    S->prof = prof;
    S->use_tc = !(flags & LEB_FLAG_FFMA_ONLY);
    S->use_pairs = S->use_tc && !(flags & LEB_FLAG_SINGLE_CTA);
    const bool cert = !(flags & LEB_FLAG_NO_MARGIN);                  // certified mode (N6): DESIGN.md §6 "Certified margin"
    const bool ibp = (flags & LEB_FLAG_IBP_HIDDEN) != 0;
    if (cert)
        for (int l = 0; l < S->L; ++l) if (S->wp[l] > 2048) return LEB_ERR_UNSUPPORTED;   // the 1.0001 norm factor covers K <= 2048
    if (tiles == 0) return LEB_OK;
    leb_status ws = ensure_workspace(S, tiles, false);
    if (ws != LEB_OK) return ws;
    const int L = S->L, n = S->w[L], N = S->w[0];
    for (int t0 = 0; t0 < tiles; t0 += S->chunk) {
        const int C = std::min(S->chunk, tiles - t0);
        pad_inputs_kernel<<<gs_grid((size_t)C * S->wp[0]), 256, 0, st>>>(C, N, ld_in, S->wp[0], nom + (size_t)t0 * ld_in,
                                                                       rad + (size_t)t0 * ld_in, S->nomp, S->radp,
                                                                       mu ? mu + (size_t)t0 * ld_in : nullptr, mu ? S->mup : nullptr);
        ++*launches;
        S->mu_cur = mu ? S->mup : nullptr;
        forward_chunk(S, C, J, J == nullptr, cert, cert && margin != nullptr, st, launches, ibp);
        size_t warps = (size_t)C * n;
        const int ks = [&] { int k = 0; for (int l = 1; l < L; ++l) k += S->wp[l]; return k; }();
        concretise_out_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>(
            C, S->rows_pad[L], n, N, S->wp[0], S->Lam[L][0], S->radp, S->gap[L], J ? J + (size_t)t0 * n * N : nullptr,
            r_lo + (size_t)t0 * ld_out, r_hi + (size_t)t0 * ld_out, ld_out, domain_flag, cert ? 1 : 0, S->marg, S->eta, S->wp[L],
            1.f + (float)(S->wp[0] + 8) * 1.1920929e-07f, 1.f + (float)(ks + 64) * 1.1920929e-07f,
            margin ? margin + (size_t)t0 * ld_out : nullptr, S->mu_cur);     // value mode: no margin is added, 0 is reported
        ++*launches;
        S->last_tiles = (tiles <= S->chunk) ? C : 0;
        S->last_with_jac = (J == nullptr);
        S->last_cert = cert;
        S->last_ibp = ibp;
        S->last_mu = (mu != nullptr);
        S->last_alpha = (S->alpha_mode == 2);
    }
    if (S->launch_failed) { S->launch_failed = false; return LEB_ERR_CUDA; }
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

void leb_nn_query(const NnState* S, int* tiles, int* certified, int* vjp_reused) {
    *tiles = S->last_tiles > 0 ? S->last_tiles : 0;
    *certified = (S->last_tiles > 0 && S->last_cert) ? 1 : 0;
    *vjp_reused = S->last_vjp_reused ? 1 : 0;
}

leb_status leb_nn_get_hidden(NnState* S, int layer, float* l, float* u, cudaStream_t st, long long* launches) {
    if (layer < 1 || layer >= S->L || S->last_tiles <= 0 || S->chunk <= 0) return LEB_ERR_STATE;
    copy_hidden_kernel<<<gs_grid((size_t)S->last_tiles * S->w[layer]), 256, 0, st>>>(S->last_tiles, S->w[layer], S->wp[layer],
                                                                                    S->lb[layer], S->ub[layer], l, u);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

// relaxation slopes (k_U, k_L) of hidden layer `layer` in the resident forward state: [tiles, dims[layer]] each
leb_status leb_nn_get_slopes(NnState* S, int layer, float* kU, float* kL, cudaStream_t st, long long* launches) {
    if (layer < 1 || layer >= S->L || S->last_tiles <= 0 || S->chunk <= 0) return LEB_ERR_STATE;
    copy_hidden_kernel<<<gs_grid((size_t)S->last_tiles * S->w[layer]), 256, 0, st>>>(S->last_tiles, S->w[layer], S->wp[layer],
                                                                                    S->kU[layer], S->kL[layer], kU, kL);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_nn_get_coeffs(NnState* S, int target, float* out, cudaStream_t st, long long* launches) {
    if (target < 2 || target > S->L || S->last_tiles <= 0 || S->chunk <= 0) return LEB_ERR_STATE;
    const int rows = S->w[target];
    copy_coeffs_kernel<<<gs_grid((size_t)S->last_tiles * 2 * rows * S->w[0]), 256, 0, st>>>(
        S->last_tiles, rows, S->rows_kind[target], S->rows_pad[target], S->w[0], S->wp[0], S->Lam[target][0], out);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

// the Jacobian chain rows J~ of the output target (rows [2 n, 3 n) of its Lambda_0 block): [tiles, n, N]
__global__ void copy_jac_kernel(int tiles, int n, int rows_pad, int N, int wp0, const float* __restrict__ Lam0, float* __restrict__ out) {
    size_t total = (size_t)tiles * n * N;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(q % N);
        size_t r = q / N;
        int i = (int)(r % n), t = (int)(r / n);
        out[q] = Lam0[((size_t)t * rows_pad + 2 * (size_t)n + i) * wp0 + c];
    }
}

leb_status leb_nn_get_jacobian(NnState* S, float* out, cudaStream_t st, long long* launches) {
    if (S->last_tiles <= 0 || S->chunk <= 0 || !S->last_with_jac) return LEB_ERR_STATE;
    const int n = S->w[S->L];
    copy_jac_kernel<<<gs_grid((size_t)S->last_tiles * n * S->w[0]), 256, 0, st>>>(S->last_tiles, n, S->rows_pad[S->L], S->w[0], S->wp[0],
                                                                               S->Lam[S->L][0], out);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------
// VJP: forward of the chunk (all coefficient blocks kept), then the reverse sweep
// ------------------------------------------------------------------------------------------
leb_status leb_nn_vjp(NnState* S, int tiles, const float* nom, const float* rad, const float* mu, const float* g_lo,
                      const float* g_hi, int ld_in, int ld_out, float* grad_nom, float* grad_rad, float* grad_mu, unsigned flags,
                      int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof) {
    (void)domain_flag;
    S->prof = prof;
    S->use_tc = !(flags & LEB_FLAG_FFMA_ONLY);
    S->use_pairs = S->use_tc && !(flags & LEB_FLAG_SINGLE_CTA);
    if (tiles == 0) return LEB_OK;
    leb_status ws = ensure_workspace(S, tiles, true);
    if (ws != LEB_OK) return ws;
    const int L = S->L, n = S->w[L], N = S->w[0], wp0 = S->wp[0];
    // LEB_FLAG_REUSE_FWD: the caller states that (nom, rad) are those of the previous leb_nn_fwd call on this context; if the
    // workspace still holds that call's complete forward state (one chunk, own Jacobian), the reverse sweep starts from it
    // and was computed in the mode this call names (LEB_FLAG_NO_MARGIN: a value-mode state; otherwise a certified one).
    const bool ibp = (flags & LEB_FLAG_IBP_HIDDEN) != 0;
    const bool want_cert = !(flags & LEB_FLAG_NO_MARGIN);
    const bool reuse = (flags & LEB_FLAG_REUSE_FWD) && S->last_tiles == tiles && S->last_with_jac && tiles <= S->chunk &&
                       S->last_cert == want_cert && S->last_ibp == ibp && S->last_mu == (mu != nullptr);
    S->last_vjp_reused = reuse;
    // a state left by leb_nn_alpha_fwd: the reverse sweep of the refined bound holds the kept slopes constant
    struct AlphaGuard { NnState* S; bool on; ~AlphaGuard() { if (on) S->alpha_mode = 0; } } alpha_guard{S, reuse && S->last_alpha && S->alpha_mode == 0};
    if (alpha_guard.on) S->alpha_mode = 2;
    for (int t0 = 0; t0 < tiles; t0 += S->chunk) {
        const int C = std::min(S->chunk, tiles - t0);
        if (!reuse)
            pad_inputs_kernel<<<gs_grid((size_t)C * wp0), 256, 0, st>>>(C, N, ld_in, wp0, nom + (size_t)t0 * ld_in,
                                                                      rad + (size_t)t0 * ld_in, S->nomp, S->radp,
                                                                      mu ? mu + (size_t)t0 * ld_in : nullptr, mu ? S->mup : nullptr);
        S->mu_cur = mu ? S->mup : nullptr;
        pad_cotangent_kernel<<<gs_grid((size_t)C * n), 256, 0, st>>>(C, n, ld_out, g_lo + (size_t)t0 * ld_out,
                                                                   g_hi + (size_t)t0 * ld_out, S->glo_p, S->ghi_p);
        *launches += 2;
        // the VJP is that of the value-mode bound: the certified margin is a rounding-level outward pad, treated as constant
        if (!reuse) forward_chunk(S, C, nullptr, true, false, false, st, launches, ibp);
        // ---- zero the adjoint accumulators
        for (int l = 1; l < L; ++l) {
            size_t c = (size_t)C * S->wp[l];
            cudaMemsetAsync(S->kUb[l], 0, c * 4, st); cudaMemsetAsync(S->kLb[l], 0, c * 4, st);
            cudaMemsetAsync(S->gUb[l], 0, c * 4, st); cudaMemsetAsync(S->gLb[l], 0, c * 4, st);
            cudaMemsetAsync(S->dpb[l], 0, c * 4, st); cudaMemsetAsync(S->zbar[l], 0, c * 4, st);
        }
        cudaMemsetAsync(S->nom_bar, 0, (size_t)C * wp0 * 4, st);
        cudaMemsetAsync(S->rad_bar, 0, (size_t)C * wp0 * 4, st);
        if (mu) cudaMemsetAsync(S->mu_bar, 0, (size_t)C * wp0 * 4, st);
        // ---- targets s = L .. 2
        for (int s = L; s >= 2; --s) {
            const bool is_out = (s == L);
            const int rp = S->rows_pad[s], rk = S->rows_kind[s], nk = is_out ? 3 : 2;
            if (!is_out) {
                relax_vjp_kernel<<<gs_grid((size_t)C * S->wp[s]), 256, 0, st>>>(S->act, C, S->w[s], S->wp[s], S->zhat[s], S->lb[s],
                                                                              S->ub[s], S->kUb[s], S->kLb[s], S->gUb[s], S->gLb[s],
                                                                              S->dpb[s], S->lbar[s], S->ubar[s], S->zbar[s], 0,
                                                                              S->alpha_mode ? S->alpha[s] : nullptr);
                ++*launches;
            }
            if (ibp && !is_out) {
                // CROWN-IBP: reverse of the interval step of layer s (see ibp_dev_kernel); mU / mL hold what layer s+1 sent
                const size_t cs = (size_t)C * S->wp[s], cp = (size_t)C * S->wp[s - 1];
                if (s < L - 1) { ibp_add_kernel<<<gs_grid(cs), 256, 0, st>>>(cs, S->lbar[s], S->ubar[s], S->zbar[s], S->mU[s], S->mL[s]); ++*launches; }
                ibp_seed_kernel<<<gs_grid(cs), 256, 0, st>>>(cs, S->lbar[s], S->ubar[s], S->cv[s], S->adev[s]);
                GemmArgs g1 = plain_args(C, S->wp[s - 1], S->wp[s], S->cv[s], S->wp[s], S->W[s], S->wp[s - 1], S->ce[s - 1], S->wp[s - 1]);
                launch_gemm<AMODE_PLAIN, EPI_STORE>(S, g1, st, launches);
                GemmArgs g2 = plain_args(C, S->wp[s - 1], S->wp[s], S->adev[s], S->wp[s], S->Wabs[s], S->wp[s - 1], S->ct[s - 1], S->wp[s - 1]);
                launch_gemm<AMODE_PLAIN, EPI_STORE>(S, g2, st, launches);
                ibp_bwd_kernel<<<gs_grid(cp), 256, 0, st>>>(S->act, C, S->w[s - 1], S->wp[s - 1], S->zhat[s - 1], S->lb[s - 1], S->ub[s - 1],
                                                           S->ce[s - 1], S->ct[s - 1], S->mU[s - 1], S->mL[s - 1], S->zbar[s - 1]);
                *launches += 2;
                continue;
            }
            const float* yu = is_out ? S->ghi_p : S->ubar[s];
            const float* yl = is_out ? S->glo_p : S->lbar[s];
            if (S->mu_cur)
                seed_kernel<true><<<dim3(C, (rk + 31) / 32), 256, 0, st>>>(is_out ? 1 : 0, rp, rk, wp0, S->Lam[s][0], S->radp, yu, yl, is_out ? n : S->wp[s],
                                                                       S->Lbar[0], S->gapbar, S->rad_bar, S->mu_cur, mu ? S->mu_bar : nullptr);
            else
                seed_kernel<false><<<dim3(C, (rk + 31) / 32), 256, 0, st>>>(is_out ? 1 : 0, rp, rk, wp0, S->Lam[s][0], S->radp, yu, yl, is_out ? n : S->wp[s],
                                                                        S->Lbar[0], S->gapbar, S->rad_bar, nullptr, nullptr);
            ++*launches;
            int cur = 0;
            for (int l = 1; l <= s - 1; ++l) {
                GemmArgs g{};
                g.M = C * rp; g.N = S->wp[l]; g.K = S->wp[l - 1];
                g.A = S->Lbar[cur]; g.lda = S->wp[l - 1];
                g.B = S->Wt[l]; g.ldb = S->rowsW[l];
                g.C = S->Lbar[cur ^ 1]; g.ldc = S->wp[l];
                g.rows_pad = rp; g.rows_kind = rk; g.nkinds = nk;
                g.kU = S->kU[l]; g.kL = S->kL[l]; g.gU = S->gU[l]; g.gL = S->gL[l]; g.dphi = S->dphi[l]; g.ldp = S->wp[l];
                g.lam_shared = (l == s - 1);
                g.Lam = g.lam_shared ? S->W[s] : S->Lam[s][l];
                g.ldl = S->wp[l];
                g.gapbar = S->gapbar;
                g.kUb = S->kUb[l]; g.kLb = S->kLb[l]; g.gUb = S->gUb[l]; g.gLb = S->gLb[l]; g.db = S->dpb[l];
                g.write_c = (l < s - 1);
                const double flops = 2.0 * C * nk * (is_out ? S->w[L] : S->w[s]) * (double)S->w[l] * S->w[l - 1];
                if (S->use_tc) {
                    S->prof->begin(LEB_KC_CHAIN_BWD, st);
                    const cudaError_t le = S->use_pairs ? tc2::launch_chain_gemm_tc2_bwd(g, S->mapW_hi[l], S->mapW_lo[l], S->num_sms, st)
                                                        : tc::launch_chain_gemm_tc<tc::MODE_BWD>(g, S->mapW_hi[l], S->mapW_lo[l], S->num_sms, st);
                    if (le != cudaSuccess) S->launch_failed = true;
                    S->prof->end(LEB_KC_CHAIN_BWD, st, flops);
                    ++*launches;
                } else {
                    launch_gemm<AMODE_PLAIN, EPI_CHAIN_BWD>(S, g, st, launches, LEB_KC_CHAIN_BWD, flops);
                }
                cur ^= 1;
            }
        }
        // ---- layer 1: l_1, u_1 = zhat_1 -+ |W_1| sigma
        relax_vjp_kernel<<<gs_grid((size_t)C * S->wp[1]), 256, 0, st>>>(S->act, C, S->w[1], S->wp[1], S->zhat[1], S->lb[1], S->ub[1],
                                                                      S->kUb[1], S->kLb[1], S->gUb[1], S->gLb[1], S->dpb[1],
                                                                      S->lbar[1], S->ubar[1], S->zbar[1], 1,
                                                                      S->alpha_mode ? S->alpha[1] : nullptr);
        if (ibp && L > 2) {
            const size_t c1 = (size_t)C * S->wp[1];
            ibp_add_kernel<<<gs_grid(c1), 256, 0, st>>>(c1, S->lbar[1], S->ubar[1], S->zbar[1], S->mU[1], S->mL[1]);
            ++*launches;
        }
        diff_kernel<<<gs_grid((size_t)C * S->wp[1]), 256, 0, st>>>(S->ubar[1], S->lbar[1], S->rad1, (size_t)C * S->wp[1]);
        *launches += 2;
        if (mu) {     // l_1, u_1 = zhat_1 + W_1 mu -+ |W_1| sigma: mu_bar += W_1^T (l_bar_1 + u_bar_1)
            sum_kernel<<<gs_grid((size_t)C * S->wp[1]), 256, 0, st>>>(S->ubar[1], S->lbar[1], S->mu1, (size_t)C * S->wp[1]);
            ++*launches;
            GemmArgs g = plain_args(C, wp0, S->wp[1], S->mu1, S->wp[1], S->W[1], wp0, S->mu_bar, wp0);
            launch_gemm<AMODE_PLAIN, EPI_ACC>(S, g, st, launches);
        }
        {
            GemmArgs g = plain_args(C, wp0, S->wp[1], S->rad1, S->wp[1], S->Wabs1, wp0, S->rad_bar, wp0);
            launch_gemm<AMODE_PLAIN, EPI_ACC>(S, g, st, launches);
        }
        // ---- nominal back-propagation: abar_{l-1} = zbar_l W_l; zbar_{l-1} += phi'(zhat_{l-1}) abar_{l-1}
        for (int l = L - 1; l >= 1; --l) {
            if (l > 1) {
                GemmArgs g = plain_args(C, S->wp[l - 1], S->wp[l], S->zbar[l], S->wp[l], S->W[l], S->wp[l - 1], S->zbar[l - 1], S->wp[l - 1]);
                g.dphi = S->dphi[l - 1]; g.ldp = S->wp[l - 1];
                launch_gemm<AMODE_PLAIN, EPI_ACC_DPHI>(S, g, st, launches);
            } else {
                GemmArgs g = plain_args(C, wp0, S->wp[1], S->zbar[1], S->wp[1], S->W[1], wp0, S->nom_bar, wp0);
                launch_gemm<AMODE_PLAIN, EPI_ACC>(S, g, st, launches);
            }
        }
        write_grads_kernel<<<gs_grid((size_t)C * N), 256, 0, st>>>(C, N, wp0, ld_in, S->nom_bar, S->rad_bar,
                                                                 grad_nom + (size_t)t0 * ld_in, grad_rad + (size_t)t0 * ld_in,
                                                                 mu ? S->mu_bar : nullptr, (mu && grad_mu) ? grad_mu + (size_t)t0 * ld_in : nullptr);
        ++*launches;
        if (!reuse) { S->last_tiles = (tiles <= S->chunk) ? C : 0; S->last_with_jac = true; S->last_cert = false; S->last_ibp = ibp; S->last_mu = (mu != nullptr); S->last_alpha = (S->alpha_mode == 2); }   // a value-mode forward state
    }
    if (S->launch_failed) { S->launch_failed = false; return LEB_ERR_CUDA; }
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------
// optimisable lower slopes (alpha-CROWN style): projected gradient descent on the lower slopes of the
// unstable ReLU neurons, one slope set per tile, objective = total width of the tile's enclosure; every iterate is sound,
// the tightest one is returned.  Forward and reverse sweep are the ordinary ones (the slope adjoints k_bar^L, gap_bar^L are
// what the reverse sweep accumulates anyway).
// ------------------------------------------------------------------------------------------
leb_status leb_nn_alpha(NnState* S, int tiles, const float* nom, const float* rad, int ld_in, int steps, float lr, float* r_lo,
                        float* r_hi, int ld_out, float* w0, float* wbest, unsigned flags, int* domain_flag, cudaStream_t st,
                        long long* launches, LebProf* prof) {
    if (S->act != ACT_RELU) return LEB_ERR_UNSUPPORTED;
    if (flags & LEB_FLAG_IBP_HIDDEN) return LEB_ERR_UNSUPPORTED;
    if (tiles == 0) return LEB_OK;
    leb_status ws = ensure_workspace(S, tiles, true);
    if (ws != LEB_OK) return ws;
    const int L = S->L, n = S->w[L];
    const size_t Cmax = (size_t)std::min(S->chunk, tiles);
    if (S->alpha_scratch_tiles < Cmax) {
        cudaDeviceSynchronize();
        for (void* p : S->alpha_scratch) cudaFree(p);
        S->alpha_scratch.clear();
        const size_t sizes[6] = {Cmax * n, Cmax * n, Cmax * n, Cmax * n, Cmax * (size_t)ld_in, Cmax * (size_t)ld_in};
        for (size_t sz : sizes) {
            void* p = nullptr;
            if (cudaMalloc(&p, std::max<size_t>(sz, 4) * sizeof(float)) != cudaSuccess) { S->alpha_scratch_tiles = 0; return LEB_ERR_NOMEM; }
            S->alpha_scratch.push_back(p);
        }
        S->alpha_scratch_tiles = Cmax;
    }
    float *cur_lo = (float*)S->alpha_scratch[0], *cur_hi = (float*)S->alpha_scratch[1], *gm1 = (float*)S->alpha_scratch[2],
          *gp1 = (float*)S->alpha_scratch[3], *gsn = (float*)S->alpha_scratch[4], *gsr = (float*)S->alpha_scratch[5];
    fill_kernel<<<gs_grid(Cmax * n), 256, 0, st>>>(gm1, Cmax * n, -1.f);
    fill_kernel<<<gs_grid(Cmax * n), 256, 0, st>>>(gp1, Cmax * n, 1.f);
    *launches += 2;
    // the descent runs on the plain (value-mode) bound; the kept slopes are then evaluated once more in the mode the caller
    // asked for -- certified by default: any slope in [0, 1] is a valid lower line, so the certificate of leb_nn_fwd carries over
    const unsigned f = flags | LEB_FLAG_NO_MARGIN;
    leb_status rc = LEB_OK;
    for (int t0 = 0; t0 < tiles && rc == LEB_OK; t0 += S->chunk) {
        const int C = std::min(S->chunk, tiles - t0);
        const float* a = nom + (size_t)t0 * ld_in;
        const float* r = rad + (size_t)t0 * ld_in;
        for (int it = 0; it <= steps && rc == LEB_OK; ++it) {
            S->alpha_mode = (it == 0) ? 1 : 2;
            rc = leb_nn_forward(S, C, a, r, nullptr, nullptr, ld_in, cur_lo, cur_hi, nullptr, n, f, domain_flag, st, launches, prof);
            if (rc != LEB_OK) break;
            alpha_best_kernel<<<C, 128, 0, st>>>(n, ld_out, it == 0 ? 1 : 0, cur_lo, cur_hi, r_lo + (size_t)t0 * ld_out, r_hi + (size_t)t0 * ld_out,
                                                 w0 + t0, wbest + t0, S->alpha_take);
            ++*launches;
            for (int l = 1; l < L; ++l) {
                alpha_keep_kernel<<<gs_grid((size_t)C * S->wp[l]), 256, 0, st>>>(C, S->wp[l], S->alpha_take, S->alpha[l], S->alpha_best[l]);
                ++*launches;
            }
            if (it == steps) break;
            S->alpha_mode = 2;
            rc = leb_nn_vjp(S, C, a, r, nullptr, gm1, gp1, ld_in, n, gsn, gsr, nullptr, f | LEB_FLAG_REUSE_FWD, domain_flag, st, launches, prof);
            if (rc != LEB_OK) break;
            for (int l = 1; l < L; ++l) {
                alpha_update_kernel<<<gs_grid((size_t)C * S->wp[l]), 256, 0, st>>>(C, S->w[l], S->wp[l], S->zhat[l], S->lb[l], S->ub[l],
                                                                                S->kLb[l], S->gLb[l], S->alpha[l], lr);
                ++*launches;
            }
        }
        if (rc != LEB_OK) break;
        // the kept slopes, in the caller's mode; the state stays resident for leb_vjp(LEB_FLAG_REUSE_FWD)
        for (int l = 1; l < L; ++l)
            cudaMemcpyAsync(S->alpha[l], S->alpha_best[l], (size_t)C * S->wp[l] * sizeof(float), cudaMemcpyDeviceToDevice, st);
        S->alpha_mode = 2;
        rc = leb_nn_forward(S, C, a, r, nullptr, nullptr, ld_in, cur_lo, cur_hi, nullptr, n, flags, domain_flag, st, launches, prof);
        if (rc != LEB_OK) break;
        alpha_best_kernel<<<C, 128, 0, st>>>(n, ld_out, 2, cur_lo, cur_hi, r_lo + (size_t)t0 * ld_out, r_hi + (size_t)t0 * ld_out, w0 + t0,
                                             wbest + t0, S->alpha_take);
        ++*launches;
    }
    S->alpha_mode = 0;
    if (tiles > S->chunk || rc != LEB_OK) S->last_tiles = 0;      // several chunks: no complete state is resident
    else S->last_tiles = tiles;
    if (rc != LEB_OK) return rc;
    return cudaGetLastError() == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

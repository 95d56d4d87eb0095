// nn_gemm_ffma.cuh -- FP32 FFMA tiled contraction with the CROWN prologue / epilogues fused in.
// This is the LEB_FLAG_FFMA_ONLY path and the path for shapes the tcgen05 kernel does not take
// (the small nominal / layer-1 / back-propagation products with M = tiles).
//
//   C[M x N] (+)= T(A)[M x K] * B[K x N]        B row-major (N contiguous), all dims multiples of 4
//
// AMODE_PLAIN : T(A) = A.
// AMODE_CHAIN : one step of the CROWN back-substitution (eq. (18); SURVEY 8(c).2
//               step 3): the A rows are coefficient rows Lambda_l of the upper / lower / Jacobian
//               chains of one tile, and the loader applies D = Lambda^+ (.) k_pos + Lambda^- (.) k_neg
//               on the fly (upper chain: (kU, kL); lower: (kL, kU); Jacobian chain: (phi', phi')) and
//               accumulates the deviation-form constant  gap += Lambda^+ . g_pos + Lambda^- . g_neg.
// EPI_*       : see the enum.
//
// Row structure of chain matrices: M = tiles * rows_pad; inside a tile, rows [0, rows_kind) are the
// upper chain, [rows_kind, 2 rows_kind) the lower chain, [2 rows_kind, 3 rows_kind) the Jacobian
// chain when nkinds == 3, the rest zero padding up to a multiple of the 128-row block.
#pragma once
#include <cuda_runtime.h>

namespace leb_nn {

enum { AMODE_PLAIN = 0, AMODE_CHAIN = 1 };
enum {
    EPI_STORE = 0,      // C = acc
    EPI_NOMINAL = 1,    // z = acc + bias; C = z; ahat = phi(z); dphi = phi'(z)
    EPI_CHAIN_BWD = 2,  // reverse chain step: mask with the forward Lambda, reduce parameter adjoints
    EPI_ACC_DPHI = 3,   // C += acc * dphi   (nominal back-propagation)
    EPI_ACC = 4         // C += acc
};

struct GemmArgs {
    int M, N, K;
    const float* A; int lda;
    const float* B; int ldb;
    float* C; int ldc;
    // chain row structure
    int rows_pad, rows_kind, nkinds, a_shared;
    // parameters of the layer on the K side (AMODE_CHAIN) or N side (EPI_CHAIN_BWD): [tiles x ldp]
    const float *kU, *kL, *gU, *gL, *dphi; int ldp;
    float* gap; int gap_init;
    // EPI_NOMINAL
    const float* bias; float* ahat; float* dphi_out; int act;
    // EPI_CHAIN_BWD
    const float* Lam; int ldl; int lam_shared; const float* gapbar;
    float *kUb, *kLb, *gUb, *gLb, *db; int write_c;
};

constexpr int BM = 128, BN = 128, BK = 16, GT = 256;

__device__ __forceinline__ void chain_row(const GemmArgs& g, int m, int& tile, int& kind, int& rk) {
    tile = m / g.rows_pad;
    int r = m - tile * g.rows_pad;
    kind = r / g.rows_kind;
    rk = r - kind * g.rows_kind;
    if (kind >= g.nkinds) kind = -1;
}

template <int AMODE, int EPI>
__global__ void __launch_bounds__(GT) gemm_ffma_kernel(GemmArgs g) {
    __shared__ __align__(16) float As[2][BK][BM + 4];
    __shared__ __align__(16) float Bs[2][BK][BN + 4];
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;

    // ---- loader coordinates
    const int a_row[2] = {tid >> 2, (tid >> 2) + 64};
    const int a_kq = (tid & 3) * 4;
    const int b_kr[2] = {tid >> 5, (tid >> 5) + 8};
    const int b_nq = (tid & 31) * 4;

    const float* a_ptr[2];
    bool a_ok[2];
    int a_kind[2] = {0, 0};
    const float *p_kpos[2] = {nullptr, nullptr}, *p_kneg[2] = {nullptr, nullptr};
    const float *p_gpos[2] = {nullptr, nullptr}, *p_gneg[2] = {nullptr, nullptr};
    const bool do_gap = (AMODE == AMODE_CHAIN) && (blockIdx.x == 0) && (g.gap != nullptr);
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        int m = m0 + a_row[i];
        a_ok[i] = m < g.M;
        a_ptr[i] = g.A;
        if (AMODE == AMODE_CHAIN) {
            int tile = 0, kind = -1, rk = 0;
            if (a_ok[i]) chain_row(g, m, tile, kind, rk);
            a_kind[i] = kind;
            if (kind < 0) a_ok[i] = false;
            else {
                a_ptr[i] = g.A + (size_t)(g.a_shared ? rk : m) * g.lda;
                size_t po = (size_t)tile * g.ldp;
                if (kind == 0) { p_kpos[i] = g.kU + po; p_kneg[i] = g.kL + po; p_gpos[i] = g.gU + po; p_gneg[i] = g.gL + po; }
                else if (kind == 1) { p_kpos[i] = g.kL + po; p_kneg[i] = g.kU + po; p_gpos[i] = g.gL + po; p_gneg[i] = g.gU + po; }
                else { p_kpos[i] = g.dphi + po; p_kneg[i] = g.dphi + po; }
            }
        } else if (a_ok[i]) {
            a_ptr[i] = g.A + (size_t)m * g.lda;
        }
    }
    float gsum[2] = {0.f, 0.f};

    float4 ra[2], rb[2];
    auto load_global = [&](int k0) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            int k = k0 + a_kq;
            ra[i] = (a_ok[i] && k < g.K) ? __ldg(reinterpret_cast<const float4*>(a_ptr[i] + k)) : make_float4(0.f, 0.f, 0.f, 0.f);
            int kr = k0 + b_kr[i], n = n0 + b_nq;
            rb[i] = (kr < g.K && n < g.N) ? __ldg(reinterpret_cast<const float4*>(g.B + (size_t)kr * g.ldb + n))
                                         : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    auto store_smem = [&](int buf, int k0) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            float4 v = ra[i];
            if (AMODE == AMODE_CHAIN) {
                int k = k0 + a_kq;
                if (a_ok[i] && k < g.K) {
                    float4 kp = __ldg(reinterpret_cast<const float4*>(p_kpos[i] + k));
                    float4 kn = __ldg(reinterpret_cast<const float4*>(p_kneg[i] + k));
                    if (do_gap && a_kind[i] < 2) {
                        float4 gp = __ldg(reinterpret_cast<const float4*>(p_gpos[i] + k));
                        float4 gn = __ldg(reinterpret_cast<const float4*>(p_gneg[i] + k));
                        gsum[i] += (v.x > 0.f ? v.x * gp.x : v.x * gn.x) + (v.y > 0.f ? v.y * gp.y : v.y * gn.y) +
                                   (v.z > 0.f ? v.z * gp.z : v.z * gn.z) + (v.w > 0.f ? v.w * gp.w : v.w * gn.w);
                    }
                    v.x = v.x > 0.f ? v.x * kp.x : v.x * kn.x;
                    v.y = v.y > 0.f ? v.y * kp.y : v.y * kn.y;
                    v.z = v.z > 0.f ? v.z * kp.z : v.z * kn.z;
                    v.w = v.w > 0.f ? v.w * kp.w : v.w * kn.w;
                }
            }
            As[buf][a_kq + 0][a_row[i]] = v.x;
            As[buf][a_kq + 1][a_row[i]] = v.y;
            As[buf][a_kq + 2][a_row[i]] = v.z;
            As[buf][a_kq + 3][a_row[i]] = v.w;
            *reinterpret_cast<float4*>(&Bs[buf][b_kr[i]][b_nq]) = rb[i];
        }
    };

    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;

    const int nk = (g.K + BK - 1) / BK;
    load_global(0);
    store_smem(0, 0);
    __syncthreads();
    for (int kt = 0; kt < nk; ++kt) {
        const int buf = kt & 1;
        if (kt + 1 < nk) load_global((kt + 1) * BK);
#pragma unroll
        for (int kk = 0; kk < BK; ++kk) {
            float4 a0 = *reinterpret_cast<const float4*>(&As[buf][kk][ty * 4]);
            float4 a1 = *reinterpret_cast<const float4*>(&As[buf][kk][64 + ty * 4]);
            float4 b0 = *reinterpret_cast<const float4*>(&Bs[buf][kk][tx * 4]);
            float4 b1 = *reinterpret_cast<const float4*>(&Bs[buf][kk][64 + tx * 4]);
            float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            float b[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        if (kt + 1 < nk) store_smem(buf ^ 1, (kt + 1) * BK);
        __syncthreads();
    }

    // ---- deviation-form constant: row sums over K, 4 loader threads per row
    if (do_gap) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            float s = gsum[i];
            s += __shfl_xor_sync(0xffffffffu, s, 1);
            s += __shfl_xor_sync(0xffffffffu, s, 2);
            int m = m0 + a_row[i];
            if ((tid & 3) == 0 && m < g.M) g.gap[m] = (g.gap_init ? 0.f : g.gap[m]) + s;
        }
    }

    // ---- epilogue
    const int rows_i[8] = {ty * 4, ty * 4 + 1, ty * 4 + 2, ty * 4 + 3, 64 + ty * 4, 65 + ty * 4, 66 + ty * 4, 67 + ty * 4};
    if (EPI == EPI_CHAIN_BWD) {
        float* red = &As[0][0][0];    // [5][BN] column partial sums (main loop is finished: reuse)
        for (int q = tid; q < 5 * BN; q += GT) red[q] = 0.f;
        __syncthreads();
        const int tile = m0 / g.rows_pad;      // blocks never straddle tiles (rows_pad % BM == 0)
        const size_t po = (size_t)tile * g.ldp;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int n = n0 + h * 64 + tx * 4;
            if (n >= g.N) continue;
            const float4 kU = *reinterpret_cast<const float4*>(g.kU + po + n), kL = *reinterpret_cast<const float4*>(g.kL + po + n);
            const float4 gU = *reinterpret_cast<const float4*>(g.gU + po + n), gL = *reinterpret_cast<const float4*>(g.gL + po + n);
            const float4 dp = *reinterpret_cast<const float4*>(g.dphi + po + n);
            float skU[4] = {0, 0, 0, 0}, skL[4] = {0, 0, 0, 0}, sgU[4] = {0, 0, 0, 0}, sgL[4] = {0, 0, 0, 0}, sdb[4] = {0, 0, 0, 0};
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int m = m0 + rows_i[i];
                if (m >= g.M) continue;
                int tl, kind, rk;
                chain_row(g, m, tl, kind, rk);
                if (kind < 0) continue;
                const float4 lam4 = *reinterpret_cast<const float4*>(g.Lam + (size_t)(g.lam_shared ? rk : m) * g.ldl + n);
                const float lam[4] = {lam4.x, lam4.y, lam4.z, lam4.w};
                const float gb = (kind < 2) ? g.gapbar[m] : 0.f;
                float out[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float Db = acc[i][h * 4 + c], lv = lam[c];
                    const float P = fmaxf(lv, 0.f), Q = fminf(lv, 0.f);
                    const float ku = (&kU.x)[c], kl = (&kL.x)[c], gu = (&gU.x)[c], gl = (&gL.x)[c], d1 = (&dp.x)[c];
                    if (kind == 0) {
                        skU[c] = fmaf(Db, P, skU[c]); skL[c] = fmaf(Db, Q, skL[c]);
                        sgU[c] = fmaf(gb, P, sgU[c]); sgL[c] = fmaf(gb, Q, sgL[c]);
                        out[c] = lv > 0.f ? fmaf(Db, ku, gb * gu) : (lv < 0.f ? fmaf(Db, kl, gb * gl) : 0.f);
                    } else if (kind == 1) {
                        skL[c] = fmaf(Db, P, skL[c]); skU[c] = fmaf(Db, Q, skU[c]);
                        sgL[c] = fmaf(gb, P, sgL[c]); sgU[c] = fmaf(gb, Q, sgU[c]);
                        out[c] = lv > 0.f ? fmaf(Db, kl, gb * gl) : (lv < 0.f ? fmaf(Db, ku, gb * gu) : 0.f);
                    } else {
                        sdb[c] = fmaf(Db, lv, sdb[c]);
                        out[c] = Db * d1;
                    }
                }
                if (g.write_c) *reinterpret_cast<float4*>(g.C + (size_t)m * g.ldc + n) = make_float4(out[0], out[1], out[2], out[3]);
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int col = h * 64 + tx * 4 + c;
                atomicAdd(&red[0 * BN + col], skU[c]);
                atomicAdd(&red[1 * BN + col], skL[c]);
                atomicAdd(&red[2 * BN + col], sgU[c]);
                atomicAdd(&red[3 * BN + col], sgL[c]);
                if (g.nkinds == 3) atomicAdd(&red[4 * BN + col], sdb[c]);
            }
        }
        __syncthreads();
        for (int q = tid; q < 5 * BN; q += GT) {
            const int a = q / BN, col = q - a * BN, n = n0 + col;
            if (n >= g.N) continue;
            if (a == 4 && g.nkinds != 3) continue;
            float* dst = (a == 0 ? g.kUb : a == 1 ? g.kLb : a == 2 ? g.gUb : a == 3 ? g.gLb : g.db) + po + n;
            atomicAdd(dst, red[q]);
        }
        return;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int m = m0 + rows_i[i];
        if (m >= g.M) continue;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int n = n0 + h * 64 + tx * 4;
            if (n >= g.N) continue;
            float4 v = make_float4(acc[i][h * 4], acc[i][h * 4 + 1], acc[i][h * 4 + 2], acc[i][h * 4 + 3]);
            float* cp = g.C + (size_t)m * g.ldc + n;
            if (EPI == EPI_STORE) {
                *reinterpret_cast<float4*>(cp) = v;
            } else if (EPI == EPI_NOMINAL) {
                const float4 bb = *reinterpret_cast<const float4*>(g.bias + n);
                v.x += bb.x; v.y += bb.y; v.z += bb.z; v.w += bb.w;
                *reinterpret_cast<float4*>(cp) = v;
                float4 a4, d4;
                if (g.act == 1) {
                    a4 = make_float4(fmaxf(v.x, 0.f), fmaxf(v.y, 0.f), fmaxf(v.z, 0.f), fmaxf(v.w, 0.f));
                    d4 = make_float4(v.x > 0.f, v.y > 0.f, v.z > 0.f, v.w > 0.f);
                } else {
                    a4 = make_float4(tanhf(v.x), tanhf(v.y), tanhf(v.z), tanhf(v.w));
                    d4 = make_float4(1.f - a4.x * a4.x, 1.f - a4.y * a4.y, 1.f - a4.z * a4.z, 1.f - a4.w * a4.w);
                }
                *reinterpret_cast<float4*>(g.ahat + (size_t)m * g.ldc + n) = a4;
                *reinterpret_cast<float4*>(g.dphi_out + (size_t)m * g.ldc + n) = d4;
            } else if (EPI == EPI_ACC_DPHI) {
                const float4 d4 = *reinterpret_cast<const float4*>(g.dphi + (size_t)m * g.ldp + n);
                float4 c4 = *reinterpret_cast<float4*>(cp);
                c4.x = fmaf(v.x, d4.x, c4.x); c4.y = fmaf(v.y, d4.y, c4.y); c4.z = fmaf(v.z, d4.z, c4.z); c4.w = fmaf(v.w, d4.w, c4.w);
                *reinterpret_cast<float4*>(cp) = c4;
            } else if (EPI == EPI_ACC) {
                float4 c4 = *reinterpret_cast<float4*>(cp);
                c4.x += v.x; c4.y += v.y; c4.z += v.z; c4.w += v.w;
                *reinterpret_cast<float4*>(cp) = c4;
            }
        }
    }
}

}  // namespace leb_nn

// tube.cu -- the consumers of the linearization-error zonotopes (Sec. IV-C, V):
//   leb_dist_add        (22) L226   r += ([E](Omega^x) (-) E_k) E_nw, the disturbance-error enclosure, in place
//   leb_tube_propagate  (27) L289   h_mu_k    = sum_{j<k} Phi_{k,j} c_bar_j
//                       (28) L291   h_sigma_k = sum_{j<k} || Phi_{k,j} E_bar_j ||_{1,r},  E_bar_j = [E  R_bar_j] (25b)
//   leb_jerr            (35) L360   J_err = sum_j sum_{k>j} || Phi_{k,j} E_bar_j ||_F^2 and d J_err / d R_bar
// E and R_bar are diagonal (L229, L519, L528, L560), so Phi E_bar = [Phi diag(E), Phi diag(R_bar)] is a column scaling:
//   h_sigma_k[i] = sum_{j<k} sum_c |Phi_{k,j}[i,c]| (|E_c| + R_bar_{j,c}),   || . ||_F^2 = sum_{i,c} Phi[i,c]^2 (E_c^2 + R_bar_{j,c}^2)
// -- no product matrix is formed.  All three are single passes over their input: HBM-bound streams (the responses Phi of
// one config-5 batch are 48 GB).  Phi is stored packed, block p(k, j) = (k-1) k / 2 + j of [T (T+1) / 2, N, n] per
// trajectory, 0 <= j < k <= T.  Widths are accumulated with every operation rounded up (they are bounds).
#include <algorithm>
#include "internal.h"

namespace {

constexpr unsigned FULL = 0xffffffffu;

// ---------------------------------------------------------------- (22)
// one warp per (tile, state i): lanes over the nw disturbance columns
__global__ void dist_add_kernel(size_t rows, int nw, const float* __restrict__ E_lo, const float* __restrict__ E_hi,
                                const float* __restrict__ E_nom, float* __restrict__ r_lo, float* __restrict__ r_hi) {
    const size_t row = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (row >= rows) return;
    const size_t o = row * (size_t)nw;
    float acc = 0.f;
    for (int j = lane; j < nw; j += 32) {
        const float e = E_nom[o + j];
        // sup |d| over d in [E_lo - e, E_hi - e], each difference rounded away from zero
        const float a = fabsf(__fadd_rd(E_lo[o + j], -e)), b = fabsf(__fadd_ru(E_hi[o + j], -e));
        acc = __fadd_ru(acc, fmaxf(fmaxf(a, b), fmaxf(fabsf(__fadd_ru(E_lo[o + j], -e)), fabsf(__fadd_rd(E_hi[o + j], -e)))));
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) acc = __fadd_ru(acc, __shfl_xor_sync(FULL, acc, off));
    if (lane == 0) {
        r_hi[row] = __fadd_ru(r_hi[row], acc);
        r_lo[row] = __fadd_rd(r_lo[row], -acc);
    }
}

// ---------------------------------------------------------------- (27)-(28)
// CTA = (trajectory b, time k, block of kRows output rows), 8 warps, each warp owns kRows / 8 rows and walks j = 0..k-1.
// The per-j vectors c_bar_j and s_j = |E| + R_bar_j are staged in shared memory (every row of the block reads them).
constexpr int kTubeWarps = 8, kRowsPerWarp = 4, kRows = kTubeWarps * kRowsPerWarp;

__global__ void __launch_bounds__(kTubeWarps * 32)
tube_kernel(int T, int n, int N, const float* __restrict__ Phi, const float* __restrict__ c_bar,
            const float* __restrict__ R_diag, const float* __restrict__ E_diag, float* __restrict__ h_mu,
            float* __restrict__ h_sigma) {
    extern __shared__ float sm[];                 // [2][2][n]: double-buffered (c_bar_j, s_j)
    const int b = blockIdx.z;
    const int k = T - (int)blockIdx.y;            // heavy (large k) CTAs first
    const int row0 = blockIdx.x * kRows;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t blocks_per_traj = (size_t)T * (T + 1) / 2;
    const float* P = Phi + ((size_t)b * blocks_per_traj + (size_t)(k - 1) * k / 2) * (size_t)N * n;
    const float* cb = c_bar + (size_t)b * T * n;
    const float* Rb = R_diag + (size_t)b * T * n;
    float mu[kRowsPerWarp], sg[kRowsPerWarp];
#pragma unroll
    for (int r = 0; r < kRowsPerWarp; ++r) { mu[r] = 0.f; sg[r] = 0.f; }
    auto stage = [&](int j, int buf) {
        float* dst = sm + (size_t)buf * 2 * n;
        for (int c = threadIdx.x; c < n; c += blockDim.x) {
            dst[c] = cb[(size_t)j * n + c];
            dst[n + c] = __fadd_ru(E_diag ? fabsf(E_diag[c]) : 0.f, Rb[(size_t)j * n + c]);
        }
    };
    stage(0, 0);
    __syncthreads();
    const bool vec = (n & 3) == 0;
    for (int j = 0; j < k; ++j) {
        if (j + 1 < k) stage(j + 1, (j + 1) & 1);
        const float* cj = sm + (size_t)(j & 1) * 2 * n;
        const float* sj = cj + n;
        const float* Pj = P + (size_t)j * N * n;
#pragma unroll
        for (int r = 0; r < kRowsPerWarp; ++r) {
            const int i = row0 + warp * kRowsPerWarp + r;
            if (i >= N) break;
            const float* row = Pj + (size_t)i * n;
            if (vec) {
                const float4* row4 = reinterpret_cast<const float4*>(row);
                for (int c4 = lane; c4 < n / 4; c4 += 32) {
                    const float4 p = __ldcs(row4 + c4);               // streamed once
                    const float4 cv = *reinterpret_cast<const float4*>(cj + 4 * c4), sv = *reinterpret_cast<const float4*>(sj + 4 * c4);
                    mu[r] = fmaf(p.x, cv.x, fmaf(p.y, cv.y, fmaf(p.z, cv.z, fmaf(p.w, cv.w, mu[r]))));
                    sg[r] = __fmaf_ru(fabsf(p.x), sv.x, __fmaf_ru(fabsf(p.y), sv.y, __fmaf_ru(fabsf(p.z), sv.z, __fmaf_ru(fabsf(p.w), sv.w, sg[r]))));
                }
            } else {
                for (int c = lane; c < n; c += 32) {
                    const float p = __ldcs(row + c);
                    mu[r] = fmaf(p, cj[c], mu[r]);
                    sg[r] = __fmaf_ru(fabsf(p), sj[c], sg[r]);
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < kRowsPerWarp; ++r) {
        float a = mu[r], s = sg[r];
#pragma unroll
        for (int off = 16; off; off >>= 1) { a += __shfl_xor_sync(FULL, a, off); s = __fadd_ru(s, __shfl_xor_sync(FULL, s, off)); }
        const int i = row0 + warp * kRowsPerWarp + r;
        if (lane == 0 && i < N) {
            const size_t o = ((size_t)b * T + (k - 1)) * N + i;
            h_mu[o] = a;
            h_sigma[o] = s;
        }
    }
}

// ---------------------------------------------------------------- (35)
// CTA = (trajectory b, disturbance index j): column energies S_c = sum_{k>j} sum_i Phi_{k,j}[i,c]^2, thread = column group,
// warps split the rows; then partial J_err of (b, j) and d J_err / d R_bar_{j,c} = 2 R_bar_{j,c} S_c.
constexpr int kJerrWarps = 8;

__global__ void __launch_bounds__(kJerrWarps * 32)
jerr_kernel(int T, int n, int N, const float* __restrict__ Phi, const float* __restrict__ R_diag,
            const float* __restrict__ E_diag, float* __restrict__ partial /* [B, T] */, float* __restrict__ grad_R) {
    extern __shared__ float sm[];                 // [kJerrWarps][n] column partials
    const int b = blockIdx.y, j = blockIdx.x;     // j ascending = heavy first
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t blocks_per_traj = (size_t)T * (T + 1) / 2;
    const float* base = Phi + (size_t)b * blocks_per_traj * (size_t)N * n;
    float* mine = sm + (size_t)warp * n;
    for (int c = lane; c < n; c += 32) mine[c] = 0.f;
    __syncwarp();
    // work items = rows of all blocks (k, j), k = j+1..T, dealt to the warps round robin
    const int nrows = (T - j) * N;
    for (int q = warp; q < nrows; q += kJerrWarps) {
        const int k = j + 1 + q / N, i = q - (k - j - 1) * N;
        const float* row = base + (((size_t)(k - 1) * k / 2 + j) * N + i) * (size_t)n;
        for (int c = lane; c < n; c += 32) { const float p = __ldcs(row + c); mine[c] = fmaf(p, p, mine[c]); }
    }
    __syncthreads();
    float acc = 0.f;
    for (int c = threadIdx.x; c < n; c += blockDim.x) {
        float S = 0.f;
#pragma unroll
        for (int w = 0; w < kJerrWarps; ++w) S += sm[(size_t)w * n + c];
        const float R = R_diag[((size_t)b * T + j) * n + c], E = E_diag ? E_diag[c] : 0.f;
        acc = fmaf(fmaf(E, E, R * R), S, acc);
        if (grad_R) grad_R[((size_t)b * T + j) * n + c] = 2.f * R * S;
    }
    __syncthreads();
#pragma unroll
    for (int off = 16; off; off >>= 1) acc += __shfl_xor_sync(FULL, acc, off);
    if (lane == 0) sm[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.f;
        for (int w = 0; w < kJerrWarps; ++w) t += sm[w];
        partial[(size_t)b * T + j] = t;
    }
}

// J_err[b] = sum_j partial[b, j], one warp per trajectory, fixed order
__global__ void jerr_finish_kernel(int B, int T, const float* __restrict__ partial, float* __restrict__ J) {
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= B) return;
    double acc = 0.0;
    for (int j = lane; j < T; j += 32) acc += (double)partial[(size_t)b * T + j];
#pragma unroll
    for (int off = 16; off; off >>= 1) acc += __shfl_xor_sync(FULL, acc, off);
    if (lane == 0) J[b] = (float)acc;
}

}  // namespace

cudaError_t leb_launch_dist_add(size_t rows, int nw, const float* E_lo, const float* E_hi, const float* E_nom, float* r_lo,
                                float* r_hi, cudaStream_t st, long long* launches, LebProf* prof) {
    if (rows == 0) return cudaSuccess;
    prof->begin(LEB_KC_TUBE, st);
    dist_add_kernel<<<(unsigned)((rows * 32 + 255) / 256), 256, 0, st>>>(rows, nw, E_lo, E_hi, E_nom, r_lo, r_hi);
    prof->end(LEB_KC_TUBE, st, 4.0 * (double)rows * (3.0 * nw + 4.0));
    ++*launches;
    return cudaGetLastError();
}

cudaError_t leb_launch_tube(int B, int T, int n, int N, const float* Phi, const float* c_bar, const float* R_diag,
                            const float* E_diag, float* h_mu, float* h_sigma, cudaStream_t st, long long* launches,
                            LebProf* prof) {
    if (B == 0 || T == 0) return cudaSuccess;
    const dim3 grid((N + kRows - 1) / kRows, T, B);
    const size_t smem = 4 * (size_t)n * sizeof(float);
    prof->begin(LEB_KC_TUBE, st);
    tube_kernel<<<grid, kTubeWarps * 32, smem, st>>>(T, n, N, Phi, c_bar, R_diag, E_diag, h_mu, h_sigma);
    // algorithmic bytes: Phi once, (c_bar, R_bar) once, two outputs
    prof->end(LEB_KC_TUBE, st, 4.0 * ((double)B * T * (T + 1) / 2 * N * n + 2.0 * B * T * n + 2.0 * B * T * N));
    ++*launches;
    return cudaGetLastError();
}

cudaError_t leb_launch_jerr(int B, int T, int n, int N, const float* Phi, const float* R_diag, const float* E_diag,
                            float* partial, float* J, float* grad_R, cudaStream_t st, long long* launches, LebProf* prof) {
    if (B == 0 || T == 0) return cudaSuccess;
    const size_t smem = std::max<size_t>((size_t)kJerrWarps * n, 32) * sizeof(float);
    prof->begin(LEB_KC_TUBE, st);
    jerr_kernel<<<dim3(T, B), kJerrWarps * 32, smem, st>>>(T, n, N, Phi, R_diag, E_diag, partial, grad_R);
    prof->end(LEB_KC_TUBE, st, 4.0 * ((double)B * T * (T + 1) / 2 * N * n + 2.0 * B * T * n));
    jerr_finish_kernel<<<(B + 7) / 8, 256, 0, st>>>(B, T, partial, J);
    *launches += 2;
    return cudaGetLastError();
}

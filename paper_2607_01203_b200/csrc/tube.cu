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
#include <mutex>
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
// One warp per output row (b, k, i): it streams the k row segments Phi_{k,j}[i, :] (n floats each) as ONE flat sequence
// of k * n / 4 16-byte items dealt round robin to the lanes -- every lane busy whatever n is -- kTubeUnroll items in
// flight per lane (the kernel is a pure HBM stream: what matters is bytes in flight), against the per-j vectors c_bar_j
// and s_j = |E| + R_bar_j, which every row of the same (b, k) re-reads from L1 / L2.
constexpr int kTubeWarps = 8, kTubeUnroll = 4;

template <bool VEC>
__global__ void __launch_bounds__(kTubeWarps * 32, 4)
tube_kernel(int T, int n, int N, const float* __restrict__ Phi, const float* __restrict__ c_bar,
            const float* __restrict__ R_diag, const float* __restrict__ E_diag, float* __restrict__ h_mu,
            float* __restrict__ h_sigma) {
    const int b = blockIdx.z;
    const int k = T - (int)blockIdx.y;            // heavy (large k) rows first
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * kTubeWarps + warp;
    if (i >= N) return;
    const size_t blocks_per_traj = (size_t)T * (T + 1) / 2;
    const float* P = Phi + (((size_t)b * blocks_per_traj + (size_t)(k - 1) * k / 2) * N + i) * (size_t)n;   // row i of Phi_{k,0}
    const size_t jstride = (size_t)N * n;
    const float* cb = c_bar + (size_t)b * T * n;
    const float* Rb = R_diag + (size_t)b * T * n;
    float mu = 0.f, sg = 0.f;
    if (VEC) {
        const int n4 = n >> 2;
        // this lane's item: (j, c4); advancing by 32 items wraps c4 over the rows
        int j = lane / n4, c4 = lane - j * n4;
        const int dj = 32 / n4, dc = 32 - dj * n4;
        // four running widths per lane (one per component): every addition is rounded up, so the excess over the exact sum
        // grows with the length of a chain -- 525 terms per lane at T = 100, n = 168 gave 1.2e-5 of the width, four chains of
        // 131 give 3e-6 -- and four independent chains instead of one serial one
        float4 sg4 = make_float4(0.f, 0.f, 0.f, 0.f);
        while (j < k) {
            float4 p[kTubeUnroll];
            int jj[kTubeUnroll], cc[kTubeUnroll];
#pragma unroll
            for (int u = 0; u < kTubeUnroll; ++u) {
                jj[u] = j; cc[u] = c4;
                if (j < k) p[u] = __ldcs(reinterpret_cast<const float4*>(P + (size_t)j * jstride) + c4);
                j += dj; c4 += dc;
                if (c4 >= n4) { c4 -= n4; ++j; }
            }
#pragma unroll
            for (int u = 0; u < kTubeUnroll; ++u) {
                if (jj[u] >= k) break;
                const float4 cv = __ldg(reinterpret_cast<const float4*>(cb + (size_t)jj[u] * n) + cc[u]);
                const float4 rv = __ldg(reinterpret_cast<const float4*>(Rb + (size_t)jj[u] * n) + cc[u]);
                const float4 e = E_diag ? __ldg(reinterpret_cast<const float4*>(E_diag) + cc[u]) : make_float4(0.f, 0.f, 0.f, 0.f);
                mu = fmaf(p[u].x, cv.x, fmaf(p[u].y, cv.y, fmaf(p[u].z, cv.z, fmaf(p[u].w, cv.w, mu))));
                sg4.x = __fmaf_ru(fabsf(p[u].x), __fadd_ru(fabsf(e.x), rv.x), sg4.x);
                sg4.y = __fmaf_ru(fabsf(p[u].y), __fadd_ru(fabsf(e.y), rv.y), sg4.y);
                sg4.z = __fmaf_ru(fabsf(p[u].z), __fadd_ru(fabsf(e.z), rv.z), sg4.z);
                sg4.w = __fmaf_ru(fabsf(p[u].w), __fadd_ru(fabsf(e.w), rv.w), sg4.w);
            }
        }
        sg = __fadd_ru(__fadd_ru(sg4.x, sg4.y), __fadd_ru(sg4.z, sg4.w));
    } else {
        for (int c = lane; c < n; c += 32) {
            const float e = E_diag ? fabsf(E_diag[c]) : 0.f;
            for (int j = 0; j < k; ++j) {
                const float p = __ldcs(P + (size_t)j * jstride + c);
                mu = fmaf(p, cb[(size_t)j * n + c], mu);
                sg = __fmaf_ru(fabsf(p), __fadd_ru(e, Rb[(size_t)j * n + c]), sg);
            }
        }
    }
#pragma unroll
    for (int off = 16; off; off >>= 1) { mu += __shfl_xor_sync(FULL, mu, off); sg = __fadd_ru(sg, __shfl_xor_sync(FULL, sg, off)); }
    if (lane == 0) {
        const size_t o = ((size_t)b * T + (k - 1)) * N + i;
        h_mu[o] = mu;
        h_sigma[o] = sg;
    }
}

// ---------------------------------------------------------------- (35)
// CTA = (trajectory b, disturbance index j): column energies S_c = sum_{k>j} sum_i Phi_{k,j}[i,c]^2.  A lane owns the
// column quads c4 = lane, lane + 32, ... (register accumulators), the warps deal the rows of all blocks (k, j),
// k = j+1..T, among themselves, kJerrUnroll rows in flight; then partial J_err of (b, j) and
// d J_err / d R_bar_{j,c} = 2 R_bar_{j,c} S_c.
constexpr int kJerrWarps = 8, kJerrQuads = 8, kJerrUnroll = 8;      // n <= 128 * kJerrQuads

template <bool VEC>
__global__ void __launch_bounds__(kJerrWarps * 32, 3)
jerr_kernel(int T, int n, int N, const float* __restrict__ Phi, const float* __restrict__ R_diag,
            const float* __restrict__ E_diag, float* __restrict__ partial /* [B, T] */, float* __restrict__ grad_R) {
    extern __shared__ float sm[];                 // [kJerrWarps][4 * ceil(n / 4)] column partials
    const int b = blockIdx.y, j = blockIdx.x;     // j ascending = heavy first
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t blocks_per_traj = (size_t)T * (T + 1) / 2;
    const float* base = Phi + (size_t)b * blocks_per_traj * (size_t)N * n;
    const int n4 = (n + 3) >> 2, nq = (n4 + 31) >> 5, np = 4 * n4;
    float4 acc[kJerrQuads];
#pragma unroll
    for (int q = 0; q < kJerrQuads; ++q) acc[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    const int nrows = (T - j) * N;
    for (int q0 = warp * kJerrUnroll; q0 < nrows; q0 += kJerrWarps * kJerrUnroll) {
        const float* row[kJerrUnroll];
#pragma unroll
        for (int u = 0; u < kJerrUnroll; ++u) {
            const int q = min(q0 + u, nrows - 1);
            const int k = j + 1 + q / N, i = q - (k - j - 1) * N;
            row[u] = base + (((size_t)(k - 1) * k / 2 + j) * N + i) * (size_t)n;
        }
#pragma unroll
        for (int cc = 0; cc < kJerrQuads; ++cc) {
            if (cc >= nq) break;
            const int c4 = lane + 32 * cc;
            float4 p[kJerrUnroll];
#pragma unroll
            for (int u = 0; u < kJerrUnroll; ++u) {
                p[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (c4 < n4 && q0 + u < nrows) {
                    if (VEC) p[u] = __ldcs(reinterpret_cast<const float4*>(row[u]) + c4);
                    else {
                        const int c = 4 * c4;
                        p[u].x = __ldcs(row[u] + c);
                        if (c + 1 < n) p[u].y = __ldcs(row[u] + c + 1);
                        if (c + 2 < n) p[u].z = __ldcs(row[u] + c + 2);
                        if (c + 3 < n) p[u].w = __ldcs(row[u] + c + 3);
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < kJerrUnroll; ++u) {
                acc[cc].x = fmaf(p[u].x, p[u].x, acc[cc].x); acc[cc].y = fmaf(p[u].y, p[u].y, acc[cc].y);
                acc[cc].z = fmaf(p[u].z, p[u].z, acc[cc].z); acc[cc].w = fmaf(p[u].w, p[u].w, acc[cc].w);
            }
        }
    }
#pragma unroll
    for (int cc = 0; cc < kJerrQuads; ++cc) {
        const int c4 = lane + 32 * cc;
        if (cc < nq && c4 < n4) reinterpret_cast<float4*>(sm + (size_t)warp * np)[c4] = acc[cc];
    }
    __syncthreads();
    float tot = 0.f;
    for (int c = threadIdx.x; c < n; c += blockDim.x) {
        float S = 0.f;
#pragma unroll
        for (int w = 0; w < kJerrWarps; ++w) S += sm[(size_t)w * np + c];
        const float R = R_diag[((size_t)b * T + j) * n + c], E = E_diag ? E_diag[c] : 0.f;
        tot = fmaf(fmaf(E, E, R * R), S, tot);
        if (grad_R) grad_R[((size_t)b * T + j) * n + c] = 2.f * R * S;
    }
    __syncthreads();
#pragma unroll
    for (int off = 16; off; off >>= 1) tot += __shfl_xor_sync(FULL, tot, off);
    if (lane == 0) sm[warp] = tot;
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
    const dim3 grid((N + kTubeWarps - 1) / kTubeWarps, T, B);
    const bool vec = (n & 3) == 0 && (((size_t)Phi | (size_t)c_bar | (size_t)R_diag | (size_t)E_diag) & 15) == 0;
    prof->begin(LEB_KC_TUBE, st);
    if (vec) tube_kernel<true><<<grid, kTubeWarps * 32, 0, st>>>(T, n, N, Phi, c_bar, R_diag, E_diag, h_mu, h_sigma);
    else tube_kernel<false><<<grid, kTubeWarps * 32, 0, st>>>(T, n, N, Phi, c_bar, R_diag, E_diag, h_mu, h_sigma);
    // algorithmic bytes: Phi once, (c_bar, R_bar) once, two outputs
    prof->end(LEB_KC_TUBE, st, 4.0 * ((double)B * T * (T + 1) / 2 * N * n + 2.0 * B * T * n + 2.0 * B * T * N));
    ++*launches;
    return cudaGetLastError();
}

cudaError_t leb_launch_jerr(int B, int T, int n, int N, const float* Phi, const float* R_diag, const float* E_diag,
                            float* partial, float* J, float* grad_R, cudaStream_t st, long long* launches, LebProf* prof) {
    if (B == 0 || T == 0) return cudaSuccess;
    const size_t smem = std::max<size_t>((size_t)kJerrWarps * 4 * ((n + 3) / 4), 32) * sizeof(float);
    const bool vec = (n & 3) == 0 && ((size_t)Phi & 15) == 0;
    prof->begin(LEB_KC_TUBE, st);
    if (vec) jerr_kernel<true><<<dim3(T, B), kJerrWarps * 32, smem, st>>>(T, n, N, Phi, R_diag, E_diag, partial, grad_R);
    else jerr_kernel<false><<<dim3(T, B), kJerrWarps * 32, smem, st>>>(T, n, N, Phi, R_diag, E_diag, partial, grad_R);
    prof->end(LEB_KC_TUBE, st, 4.0 * ((double)B * T * (T + 1) / 2 * N * n + 2.0 * B * T * n));
    jerr_finish_kernel<<<(B + 7) / 8, 256, 0, st>>>(B, T, partial, J);
    *launches += 2;
    return cudaGetLastError();
}

// ---------------------------------------------------------------- leb_jerr_static: (35) with no allocation anywhere
// The per-(b, j) partial sums of jerr_kernel -- the one scratch buffer leb_jerr takes from cudaMalloc -- live in a
// file-scope device array instead: LEB_JERR_STATIC_MAX floats (256 KB), held by every GPU that loads the library until the
// process exits.  In host code the name g_jerr_partial is only a stand-in for the symbol, not a device address: the
// address is resolved once per device, at set-up (leb_create), with that device current, and that pointer is what the
// kernels are given.  Nothing in the array has to start at zero -- jerr_kernel writes every entry (b, j) that
// jerr_finish_kernel reads, in the same call -- and it keeps the last call's contents; all calls on a device share it, so
// two calls that overlap on the GPU (different streams) race.
static __device__ __align__(256) float g_jerr_partial[LEB_JERR_STATIC_MAX];

namespace {
constexpr int kMaxDevices = 64;
float* g_jerr_partial_ptr[kMaxDevices] = {nullptr};
std::mutex g_jerr_setup_mutex;
}  // namespace

// set-up: called by leb_create with `device` current
cudaError_t leb_jerr_static_setup(int device) {
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_jerr_setup_mutex);
    if (g_jerr_partial_ptr[device]) return cudaSuccess;
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_jerr_partial);
    if (e != cudaSuccess) return e;
    g_jerr_partial_ptr[device] = static_cast<float*>(p);
    return cudaSuccess;
}

// the two launches of leb_launch_jerr on the static scratch: no allocation, no event, no profiling hook
cudaError_t leb_launch_jerr_static(int device, int B, int T, int n, int N, const float* Phi, const float* R_diag, const float* E_diag,
                                   float* J, float* grad_R, cudaStream_t st, long long* launches) {
    if (B == 0 || T == 0) return cudaSuccess;
    if (device < 0 || device >= kMaxDevices || !g_jerr_partial_ptr[device]) return cudaErrorNotReady;   // set-up did not run or failed
    if ((long long)B * T > (long long)LEB_JERR_STATIC_MAX) return cudaErrorInvalidValue;
    float* partial = g_jerr_partial_ptr[device];
    const size_t smem = std::max<size_t>((size_t)kJerrWarps * 4 * ((n + 3) / 4), 32) * sizeof(float);
    const bool vec = (n & 3) == 0 && ((size_t)Phi & 15) == 0;
    if (vec) jerr_kernel<true><<<dim3(T, B), kJerrWarps * 32, smem, st>>>(T, n, N, Phi, R_diag, E_diag, partial, grad_R);
    else jerr_kernel<false><<<dim3(T, B), kJerrWarps * 32, smem, st>>>(T, n, N, Phi, R_diag, E_diag, partial, grad_R);
    jerr_finish_kernel<<<(B + 7) / 8, 256, 0, st>>>(B, T, partial, J);
    *launches += 2;
    return cudaGetLastError();
}

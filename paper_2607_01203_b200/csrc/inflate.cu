// inflate.cu -- leb_zonotope_inflate: fold [r_lo, r_hi] into the non-zero-centred disturbance
// zonotope (c_bar, R_bar) of PAPER.md:L229-231, E_bar = [E  R_bar] of (25b) L277, with the small
// positive diagonal padding of L347.  Pure HBM stream: float4 loads/stores, grid-stride, no smem.
//
// Rounding: c = RN((lo + hi)/2); R = RU(max(hi - c, c - lo)) + pad (RU), so that in FP32
// [lo, hi] is inside [c - R, c + R].
#include "internal.h"

namespace {

__device__ __forceinline__ void fold1(float lo, float hi, float pad, float& c, float& R) {
    c = 0.5f * lo + 0.5f * hi;                       // exact halves, one rounding in the add
    float a = __fadd_ru(hi, -c), b = __fadd_ru(c, -lo);
    R = __fadd_ru(fmaxf(a, b), pad);
}

__global__ void inflate_kernel(size_t count, const float* __restrict__ r_lo, const float* __restrict__ r_hi, float pad,
                               float* __restrict__ c_bar, float* __restrict__ R_diag, int vec) {
    size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec) {
        size_t n4 = count / 4;
        const float4* lo4 = reinterpret_cast<const float4*>(r_lo);
        const float4* hi4 = reinterpret_cast<const float4*>(r_hi);
        float4* c4 = reinterpret_cast<float4*>(c_bar);
        float4* R4 = reinterpret_cast<float4*>(R_diag);
        for (size_t q = i; q < n4; q += stride) {
            float4 lo = __ldg(lo4 + q), hi = __ldg(hi4 + q), c, R;
            fold1(lo.x, hi.x, pad, c.x, R.x);
            fold1(lo.y, hi.y, pad, c.y, R.y);
            fold1(lo.z, hi.z, pad, c.z, R.z);
            fold1(lo.w, hi.w, pad, c.w, R.w);
            c4[q] = c;
            R4[q] = R;
        }
        for (size_t q = n4 * 4 + i; q < count; q += stride) fold1(r_lo[q], r_hi[q], pad, c_bar[q], R_diag[q]);
    } else {
        for (size_t q = i; q < count; q += stride) fold1(r_lo[q], r_hi[q], pad, c_bar[q], R_diag[q]);
    }
}

// dense E_bar rows: row (tile, i) is 2n floats: E_diag[i] at column i, R_diag at column n + i, zeros elsewhere.
// One thread per float4 of the output (n even and 2n % 4 == 0 handled by the scalar fallback otherwise).
__global__ void ebar_kernel(size_t rows, int n, const float* __restrict__ R_diag, const float* __restrict__ E_diag,
                            float* __restrict__ Ebar, int vec) {
    size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int w = 2 * n;
    if (vec) {
        const int w4 = w / 4;
        size_t total = rows * (size_t)w4;
        float4* out = reinterpret_cast<float4*>(Ebar);
        for (size_t q = i0; q < total; q += stride) {
            size_t row = q / w4;
            int c0 = (int)(q - row * w4) * 4;
            int i = (int)(row % n);
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            int ce = i - c0, cr = n + i - c0;
            float e = E_diag ? E_diag[i] : 0.f;
            if (ce >= 0 && ce < 4) (&v.x)[ce] = e;
            if (cr >= 0 && cr < 4) (&v.x)[cr] = R_diag[row];
            __stcs(out + q, v);   // streaming store: written once, never re-read here
        }
    } else {
        size_t total = rows * (size_t)w;
        for (size_t q = i0; q < total; q += stride) {
            size_t row = q / w;
            int c = (int)(q - row * w);
            int i = (int)(row % n);
            float v = 0.f;
            if (c == i) v = E_diag ? E_diag[i] : 0.f;
            else if (c == n + i) v = R_diag[row];
            Ebar[q] = v;
        }
    }
}

__global__ void inflate_vjp_kernel(size_t count, const float* __restrict__ gc, const float* __restrict__ gR,
                                   float* __restrict__ g_lo, float* __restrict__ g_hi) {
    size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < count; q += stride) {
        float c = gc[q], r = gR[q];
        g_lo[q] = 0.5f * c - 0.5f * r;
        g_hi[q] = 0.5f * c + 0.5f * r;
    }
}

inline bool al16(const void* p) { return ((size_t)p & 15) == 0; }
inline unsigned grid_for(size_t work, int threads) {
    size_t b = (work + threads - 1) / threads;
    size_t cap = 148 * 16;   // 148 SMs x 16 resident 256-thread CTAs: grid-stride beyond that
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned)b;
}

}  // namespace

cudaError_t leb_launch_inflate(size_t rows, int n, const float* r_lo, const float* r_hi, const float* E_diag, float pad,
                               float* c_bar, float* R_diag, float* Ebar_dense, cudaStream_t st, long long* launches,
                               LebProf* prof) {
    if (rows == 0) return cudaSuccess;
    int vec = al16(r_lo) && al16(r_hi) && al16(c_bar) && al16(R_diag);
    size_t work = vec ? rows / 4 + 1 : rows;
    prof->begin(LEB_KC_INFLATE, st);
    inflate_kernel<<<grid_for(work, 256), 256, 0, st>>>(rows, r_lo, r_hi, pad, c_bar, R_diag, vec);
    prof->end(LEB_KC_INFLATE, st, 16.0 * (double)rows);   // algorithmic bytes: 2 arrays in, 2 out
    ++*launches;
    if (Ebar_dense) {
        int v2 = al16(Ebar_dense) && ((2 * n) % 4 == 0);
        size_t w2 = v2 ? rows * (size_t)(2 * n / 4) : rows * (size_t)(2 * n);
        prof->begin(LEB_KC_INFLATE, st);
        ebar_kernel<<<grid_for(w2, 256), 256, 0, st>>>(rows, n, R_diag, E_diag, Ebar_dense, v2);
        prof->end(LEB_KC_INFLATE, st, 4.0 * (double)rows * (2.0 * n + 1.0));
        ++*launches;
    }
    return cudaGetLastError();
}

cudaError_t leb_launch_inflate_vjp(size_t count, const float* gc, const float* gR, float* g_lo, float* g_hi,
                                   cudaStream_t st, long long* launches) {
    if (count == 0) return cudaSuccess;
    inflate_vjp_kernel<<<grid_for(count, 256), 256, 0, st>>>(count, gc, gR, g_lo, g_hi);
    ++*launches;
    return cudaGetLastError();
}

// nn_gemm_tc.cuh -- the CROWN chain contraction on the 5th-generation tensor cores (tcgen05), 3xTF32.
//
// One step of the back-substitution (eq. (18)) and one step of
// its reverse sweep are dense contractions  C[M x N] = T(A)[M x K] * B[K x N]  with
// M = tiles * rows (10^5 .. 10^6), K, N = layer widths, and B a weight matrix shared by all tiles.
// FP32 operands are split  x = hi + lo  (hi = tf32(x), lo = tf32(x - hi)) and the product is
// accumulated in FP32 in tensor memory as  Ahi*Bhi + Ahi*Blo + Alo*Bhi  (the dropped Alo*Blo term and
// the rounding of lo are <= 3 * 2^-22 |a||b| per product).
//
// Kernel layout (persistent, one CTA per SM, 384 threads):
//   warp 0      TMA producer: pre-split weight tiles Bhi, Blo [256 x 32] (K-major, 128B swizzle)
//   warp 1      MMA issuer: 12 tcgen05.mma (M128 x N<=256 x K8) per 32-wide K slab, accumulators in TMEM
//   warp 2      TMEM allocation (2 x 256 columns: the epilogue of tile i overlaps the main loop of i+1)
//   warps 4-7   epilogue: tcgen05.ld -> registers -> global (forward: Lambda_{l-1};
//               reverse: sign-masked adjoint + column sums of the relaxation-parameter adjoints)
//   warps 8-11  A producers: global FP32 rows -> (forward: D = Lam^+ k_pos + Lam^- k_neg and the
//               deviation-form constant  gap += Lam^+ g_pos + Lam^- g_neg) -> hi/lo split ->
//               128B-swizzled K-major shared-memory tiles (generic-proxy stores + async-proxy fence)
// Stages are handed over with mbarriers: full[s] (128 producer arrivals + the TMA transaction),
// empty[s] (tcgen05.commit), tmem_full[a] (tcgen05.commit), tmem_empty[a] (128 epilogue arrivals).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "nn_gemm_ffma.cuh"

namespace leb_nn {
namespace tc {

enum { MODE_FWD = 0, MODE_BWD = 1 };

constexpr int TBM = 128, TBN = 256, TBK = 32, STAGES = 2;
constexpr int A_TILE_BYTES = TBM * TBK * 4;                         // 16 KB
constexpr int B_TILE_BYTES = TBN * TBK * 4;                         // 32 KB
constexpr int STAGE_BYTES = 2 * A_TILE_BYTES + 2 * B_TILE_BYTES;    // 96 KB
constexpr int RED_BYTES = 5 * TBN * 4;                              // reverse epilogue column sums
constexpr int BAR_BYTES = 128;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + RED_BYTES + BAR_BYTES + 1024;   // + 1024-byte alignment slack
constexpr int THREADS = 384;
constexpr int TMEM_COLS = 512;
constexpr unsigned long long kSpinLimit = 4000000000ull;            // ~2 s of SM clocks: trap instead of hanging

// ---------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    if (mbar_try_wait(bar, parity)) return;
    const long long t0 = clock64();
    while (!mbar_try_wait(bar, parity)) {
        if ((unsigned long long)(clock64() - t0) > kSpinLimit) __trap();   // never hang the GPU
    }
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem], kind::tf32, issued by one thread
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// 32 lanes x 32 columns of FP32: thread t of the warp gets lane (warp%4)*32 + t, columns [c, c+32)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float* v) {
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float to_tf32(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }

// K-major, 128B-swizzled operand tile: rows of 128 bytes, 8-row groups 1024 bytes apart
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);        // start address, bits [0,14)
    d |= (uint64_t)1 << 16;                          // leading byte offset (unused for swizzled K-major), bits [16,30)
    d |= (uint64_t)(1024 >> 4) << 32;                // stride byte offset: 8 rows x 128 B, bits [32,46)
    d |= (uint64_t)1 << 46;                          // descriptor version (Blackwell), bits [46,48)
    d |= (uint64_t)2 << 61;                          // layout: SWIZZLE_128B, bits [61,64)
    return d;
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, dense
__device__ __forceinline__ uint32_t make_idesc(int mma_m, int mma_n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(mma_n >> 3) << 17) | ((uint32_t)(mma_m >> 4) << 24);
}

// butterfly transpose-reduce: on return v[0] of lane L holds sum over the warp's lanes of v[L]
__device__ __forceinline__ void warp_transpose_sum32(float* v, int lane) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const bool up = (lane & off) != 0;
#pragma unroll
        for (int j = 0; j < off; ++j) {
            const float send = up ? v[j] : v[j + off];
            const float keep = up ? v[j + off] : v[j];
            v[j] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(THREADS, 1)
chain_gemm_tc_kernel(const GemmArgs g, const __grid_constant__ CUtensorMap tm_hi, const __grid_constant__ CUtensorMap tm_lo) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* sgen = smem_raw + (sbase - smem_u32(smem_raw));           // generic pointer to the aligned base
    // stage s: [Ahi | Alo | Bhi | Blo]
    auto sA = [&](int s, int part) { return sbase + s * STAGE_BYTES + part * A_TILE_BYTES; };
    auto sB = [&](int s, int part) { return sbase + s * STAGE_BYTES + 2 * A_TILE_BYTES + part * B_TILE_BYTES; };
    float* s_red = reinterpret_cast<float*>(sgen + STAGES * STAGE_BYTES);
    const uint32_t bar0 = sbase + STAGES * STAGE_BYTES + RED_BYTES;
    auto bar_full = [&](int s) { return bar0 + 8 * s; };
    auto bar_empty = [&](int s) { return bar0 + 8 * (STAGES + s); };
    auto bar_tfull = [&](int a) { return bar0 + 8 * (2 * STAGES + a); };
    auto bar_tempty = [&](int a) { return bar0 + 8 * (2 * STAGES + 2 + a); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sgen + STAGES * STAGE_BYTES + RED_BYTES + 8 * (2 * STAGES + 4));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_blocks = (g.N + TBN - 1) / TBN;
    const int m_blocks = g.M / TBM;
    const int num_tiles = m_blocks * n_blocks;
    const int nk = g.K / TBK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_hi);
        tma_prefetch_desc(&tm_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full(s), 128 + 1); mbar_init(bar_empty(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(bar_tfull(a), 1); mbar_init(bar_tempty(a), 128); }
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===================== TMA producer (weights) =====================
        int stage = 0; uint32_t phase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            const int n0 = (tile % n_blocks) * TBN;
            for (int kt = 0; kt < nk; ++kt) {
                mbar_wait(bar_empty(stage), phase ^ 1);
                if (lane == 0) {
                    mbar_arrive_expect_tx(bar_full(stage), 2 * B_TILE_BYTES);
                    tma_load_2d(sB(stage, 0), &tm_hi, kt * TBK, n0, bar_full(stage));
                    tma_load_2d(sB(stage, 1), &tm_lo, kt * TBK, n0, bar_full(stage));
                }
                __syncwarp();
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        int stage = 0; uint32_t phase = 0;
        int tcount = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcount) {
            const int n0 = (tile % n_blocks) * TBN;
            const int n_mma = min(TBN, g.N - n0);
            const uint32_t idesc = make_idesc(TBM, n_mma);
            const int acc = tcount & 1;
            mbar_wait(bar_tempty(acc), ((tcount >> 1) & 1) ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * TBN;
            for (int kt = 0; kt < nk; ++kt) {
                mbar_wait(bar_full(stage), phase);
                tc_fence_after();
                if (lane == 0) {
                    const uint64_t ahi = make_smem_desc(sA(stage, 0)), alo = make_smem_desc(sA(stage, 1));
                    const uint64_t bhi = make_smem_desc(sB(stage, 0)), blo = make_smem_desc(sB(stage, 1));
#pragma unroll
                    for (int k = 0; k < TBK / 8; ++k) {
                        const uint64_t ko = (uint64_t)(k * 32 >> 4);     // 8 tf32 = 32 bytes along K inside the swizzle atom
                        umma_tf32(d_tmem, alo + ko, bhi + ko, idesc, (kt | k) != 0);
                        umma_tf32(d_tmem, ahi + ko, blo + ko, idesc, 1u);
                        umma_tf32(d_tmem, ahi + ko, bhi + ko, idesc, 1u);
                    }
                    umma_commit(bar_empty(stage));                       // frees the stage when these MMAs retire
                    if (kt == nk - 1) umma_commit(bar_tfull(acc));       // accumulator complete
                }
                __syncwarp();
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== epilogue =====================
        const int q = warp - 4;                    // TMEM lane quadrant of this warp (warp % 4)
        const int etid = threadIdx.x - 128;
        int tcount = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcount) {
            const int mb = tile / n_blocks, n0 = (tile - mb * n_blocks) * TBN;
            const int n_mma = min(TBN, g.N - n0);
            const int acc = tcount & 1;
            const int m = mb * TBM + q * 32 + lane;
            int tl = 0, kind = 0, rk = 0;
            chain_row(g, m, tl, kind, rk);
            const size_t po = (size_t)tl * g.ldp;
            if (MODE == MODE_BWD) {
                for (int i = etid; i < 5 * TBN; i += 128) s_red[i] = 0.f;
                named_bar_sync(1, 128);
            }
            mbar_wait(bar_tfull(acc), (tcount >> 1) & 1);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + acc * TBN;
            if (MODE == MODE_FWD) {
                float* crow = g.C + (size_t)m * g.ldc + n0;
                for (int c = 0; c < n_mma; c += 32) {
                    float v[32];
                    tmem_ld32(taddr + c, v);
#pragma unroll
                    for (int j = 0; j < 32; j += 4)
                        *reinterpret_cast<float4*>(crow + c + j) = make_float4(v[j], v[j + 1], v[j + 2], v[j + 3]);
                }
            } else {
                const float gb = (kind >= 0 && kind < 2) ? g.gapbar[m] : 0.f;
                const float* lrow = g.Lam + (size_t)(g.lam_shared ? rk : m) * g.ldl + n0;
                float* crow = g.C + (size_t)m * g.ldc + n0;
                for (int c = 0; c < n_mma; c += 32) {
                    float v[32], lam[32], t[32];
                    tmem_ld32(taddr + c, v);
#pragma unroll
                    for (int j = 0; j < 32; j += 4) {
                        const float4 x = (kind >= 0) ? __ldg(reinterpret_cast<const float4*>(lrow + c + j)) : make_float4(0.f, 0.f, 0.f, 0.f);
                        lam[j] = x.x; lam[j + 1] = x.y; lam[j + 2] = x.z; lam[j + 3] = x.w;
                    }
#pragma unroll
                    for (int j = 0; j < 32; ++j) v[j] = (kind >= 0) ? v[j] : 0.f;     // padding rows may hold anything
                    // ---- column sums over the rows of this warp, one adjoint at a time (register pressure)
                    // kUb: upper rows Db*P, lower rows Db*Q;  kLb: the other way round
#pragma unroll
                    for (int j = 0; j < 32; ++j) t[j] = (kind == 0) ? v[j] * fmaxf(lam[j], 0.f) : ((kind == 1) ? v[j] * fminf(lam[j], 0.f) : 0.f);
                    warp_transpose_sum32(t, lane);
                    atomicAdd(&s_red[0 * TBN + c + lane], t[0]);
#pragma unroll
                    for (int j = 0; j < 32; ++j) t[j] = (kind == 0) ? v[j] * fminf(lam[j], 0.f) : ((kind == 1) ? v[j] * fmaxf(lam[j], 0.f) : 0.f);
                    warp_transpose_sum32(t, lane);
                    atomicAdd(&s_red[1 * TBN + c + lane], t[0]);
                    // gUb / gLb: the same with the row's gap adjoint in place of Db
#pragma unroll
                    for (int j = 0; j < 32; ++j) t[j] = (kind == 0) ? gb * fmaxf(lam[j], 0.f) : ((kind == 1) ? gb * fminf(lam[j], 0.f) : 0.f);
                    warp_transpose_sum32(t, lane);
                    atomicAdd(&s_red[2 * TBN + c + lane], t[0]);
#pragma unroll
                    for (int j = 0; j < 32; ++j) t[j] = (kind == 0) ? gb * fminf(lam[j], 0.f) : ((kind == 1) ? gb * fmaxf(lam[j], 0.f) : 0.f);
                    warp_transpose_sum32(t, lane);
                    atomicAdd(&s_red[3 * TBN + c + lane], t[0]);
                    if (g.nkinds == 3) {       // Jacobian chain: adjoint of phi'(zhat)
#pragma unroll
                        for (int j = 0; j < 32; ++j) t[j] = (kind == 2) ? v[j] * lam[j] : 0.f;
                        warp_transpose_sum32(t, lane);
                        atomicAdd(&s_red[4 * TBN + c + lane], t[0]);
                    }
                    // ---- the masked adjoint of Lambda_l
                    if (g.write_c) {
                        const float* pk = (kind == 0 ? g.kU : (kind == 1 ? g.kL : g.dphi)) + po + n0 + c;   // slope on Lam > 0
                        const float* nk_ = (kind == 0 ? g.kL : (kind == 1 ? g.kU : g.dphi)) + po + n0 + c;  // slope on Lam < 0
                        const float* pg = (kind == 0 ? g.gU : g.gL) + po + n0 + c;
                        const float* ng = (kind == 0 ? g.gL : g.gU) + po + n0 + c;
                        const float gbe = (kind == 2) ? 0.f : gb;
#pragma unroll
                        for (int j = 0; j < 32; j += 4) {
                            const float4 kp = __ldg(reinterpret_cast<const float4*>(pk + j)), kn = __ldg(reinterpret_cast<const float4*>(nk_ + j));
                            const float4 gp = __ldg(reinterpret_cast<const float4*>(pg + j)), gn = __ldg(reinterpret_cast<const float4*>(ng + j));
                            float4 o;
                            o.x = lam[j] > 0.f ? fmaf(v[j], kp.x, gbe * gp.x) : (lam[j] < 0.f ? fmaf(v[j], kn.x, gbe * gn.x) : 0.f);
                            o.y = lam[j + 1] > 0.f ? fmaf(v[j + 1], kp.y, gbe * gp.y) : (lam[j + 1] < 0.f ? fmaf(v[j + 1], kn.y, gbe * gn.y) : 0.f);
                            o.z = lam[j + 2] > 0.f ? fmaf(v[j + 2], kp.z, gbe * gp.z) : (lam[j + 2] < 0.f ? fmaf(v[j + 2], kn.z, gbe * gn.z) : 0.f);
                            o.w = lam[j + 3] > 0.f ? fmaf(v[j + 3], kp.w, gbe * gp.w) : (lam[j + 3] < 0.f ? fmaf(v[j + 3], kn.w, gbe * gn.w) : 0.f);
                            if (kind == 2) {   // Jacobian chain: Db * phi' irrespective of the sign of Lam (FFMA path: out = Db * d1)
                                o.x = v[j] * kp.x; o.y = v[j + 1] * kp.y; o.z = v[j + 2] * kp.z; o.w = v[j + 3] * kp.w;
                            }
                            if (kind < 0) o = make_float4(0.f, 0.f, 0.f, 0.f);
                            *reinterpret_cast<float4*>(crow + c + j) = o;
                        }
                    }
                }
            }
            // release the accumulator to the MMA warp
            tc_fence_before();
            mbar_arrive(bar_tempty(acc));
            if (MODE == MODE_BWD) {
                named_bar_sync(1, 128);
                const int nq = (g.nkinds == 3) ? 5 : 4;
                for (int i = etid; i < nq * TBN; i += 128) {
                    const int a = i / TBN, col = i - a * TBN;
                    if (col >= n_mma) continue;
                    float* dst = (a == 0 ? g.kUb : a == 1 ? g.kLb : a == 2 ? g.gUb : a == 3 ? g.gLb : g.db) + po + n0 + col;
                    atomicAdd(dst, s_red[i]);
                }
                named_bar_sync(1, 128);
            }
        }
    } else if (warp >= 8) {
        // ===================== A producers =====================
        const int ptid = threadIdx.x - 256, pw = ptid >> 5;
        const int r4 = lane >> 3, c4 = lane & 7;
        int stage = 0; uint32_t phase = 0;
        const float* aptr[8];
        uint32_t kinds_cur = 0, kinds_nxt = 0;
        size_t po_cur = 0, po_nxt = 0;
        int m0_cur = 0, m0_nxt = 0, nb_cur = 0, nb_nxt = 0;
        float4 cur[8], nxt[8];
        auto setup_tile = [&](int tile, uint32_t& kinds, size_t& po, int& m0, int& nb) {
            const int mb = tile / n_blocks;
            nb = tile - mb * n_blocks;
            m0 = mb * TBM;
            kinds = 0;
            int tl = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int m = m0 + pw * 32 + i * 4 + r4;
                int kind = 0, rk = 0;
                if (MODE == MODE_FWD) {
                    chain_row(g, m, tl, kind, rk);
                    if (kind < 0) { kind = 3; rk = 0; }
                    aptr[i] = g.A + (size_t)(g.a_shared ? rk : m) * g.lda + c4 * 4;
                } else {
                    aptr[i] = g.A + (size_t)m * g.lda + c4 * 4;
                }
                kinds |= (uint32_t)kind << (2 * i);
            }
            po = (size_t)(m0 / g.rows_pad) * g.ldp;
        };
        auto load_slab = [&](float4* dst, uint32_t kinds, int kt) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const bool ok = ((kinds >> (2 * i)) & 3u) != 3u;
                dst[i] = ok ? __ldg(reinterpret_cast<const float4*>(aptr[i] + kt * TBK)) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        };
        int tile = blockIdx.x, kt = 0;
        bool have = tile < num_tiles;
        if (have) {
            setup_tile(tile, kinds_cur, po_cur, m0_cur, nb_cur);
            load_slab(cur, kinds_cur, 0);
        }
        float gsum[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) gsum[i] = 0.f;
        while (have) {
            // ---- prefetch the next slab (possibly of the next tile) into registers
            int ntile = tile, nkt = kt + 1;
            if (nkt == nk) { nkt = 0; ntile = tile + gridDim.x; }
            const bool nhave = ntile < num_tiles;
            kinds_nxt = kinds_cur; po_nxt = po_cur; m0_nxt = m0_cur; nb_nxt = nb_cur;
            if (nhave) {
                if (nkt == 0) setup_tile(ntile, kinds_nxt, po_nxt, m0_nxt, nb_nxt);
                load_slab(nxt, kinds_nxt, nkt);
            }
            // ---- transform + split the current slab into the stage
            const int col = kt * TBK + c4 * 4;
            float4 kU4 = make_float4(0.f, 0.f, 0.f, 0.f), kL4 = kU4, dp4 = kU4, gU4 = kU4, gL4 = kU4;
            const bool do_gap = (MODE == MODE_FWD) && (nb_cur == 0) && (g.gap != nullptr);
            if (MODE == MODE_FWD) {
                kU4 = __ldg(reinterpret_cast<const float4*>(g.kU + po_cur + col));
                kL4 = __ldg(reinterpret_cast<const float4*>(g.kL + po_cur + col));
                if (g.nkinds == 3) dp4 = __ldg(reinterpret_cast<const float4*>(g.dphi + po_cur + col));
                if (do_gap) {
                    gU4 = __ldg(reinterpret_cast<const float4*>(g.gU + po_cur + col));
                    gL4 = __ldg(reinterpret_cast<const float4*>(g.gL + po_cur + col));
                }
            }
            mbar_wait(bar_empty(stage), phase ^ 1);
            const uint32_t a_hi = sA(stage, 0), a_lo = sA(stage, 1);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                float4 v = cur[i];
                if (MODE == MODE_FWD) {
                    const uint32_t kind = (kinds_cur >> (2 * i)) & 3u;
                    const float4 kp = kind == 0 ? kU4 : (kind == 1 ? kL4 : dp4);
                    const float4 kn = kind == 0 ? kL4 : (kind == 1 ? kU4 : dp4);
                    if (do_gap && kind < 2) {
                        const float4 gp = kind == 0 ? gU4 : gL4, gn = kind == 0 ? gL4 : gU4;
                        gsum[i] += (v.x > 0.f ? v.x * gp.x : v.x * gn.x) + (v.y > 0.f ? v.y * gp.y : v.y * gn.y) +
                                   (v.z > 0.f ? v.z * gp.z : v.z * gn.z) + (v.w > 0.f ? v.w * gp.w : v.w * gn.w);
                    }
                    if (kind != 3u) {
                        v.x = v.x > 0.f ? v.x * kp.x : v.x * kn.x;
                        v.y = v.y > 0.f ? v.y * kp.y : v.y * kn.y;
                        v.z = v.z > 0.f ? v.z * kp.z : v.z * kn.z;
                        v.w = v.w > 0.f ? v.w * kp.w : v.w * kn.w;
                    }
                }
                float4 hi, lo;
                hi.x = to_tf32(v.x); hi.y = to_tf32(v.y); hi.z = to_tf32(v.z); hi.w = to_tf32(v.w);
                lo.x = to_tf32(v.x - hi.x); lo.y = to_tf32(v.y - hi.y); lo.z = to_tf32(v.z - hi.z); lo.w = to_tf32(v.w - hi.w);
                const int row = pw * 32 + i * 4 + r4;
                const uint32_t off = (uint32_t)row * 128u + (uint32_t)((c4 ^ (row & 7)) << 4);
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a_hi + off), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w) : "memory");
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a_lo + off), "f"(lo.x), "f"(lo.y), "f"(lo.z), "f"(lo.w) : "memory");
            }
            fence_proxy_async();                 // generic-proxy stores -> visible to the tensor core's async proxy
            mbar_arrive(bar_full(stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
            // ---- end of a tile: the deviation-form constant (row sums over K; 8 threads per row)
            if (kt == nk - 1) {
                if (do_gap) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        float s = gsum[i];
                        s += __shfl_xor_sync(0xffffffffu, s, 1);
                        s += __shfl_xor_sync(0xffffffffu, s, 2);
                        s += __shfl_xor_sync(0xffffffffu, s, 4);
                        const int m = m0_cur + pw * 32 + i * 4 + r4;
                        if (c4 == 0) g.gap[m] = (g.gap_init ? 0.f : g.gap[m]) + s;
                    }
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) gsum[i] = 0.f;
            }
            // ---- advance
            tile = ntile; kt = nkt; have = nhave;
            kinds_cur = kinds_nxt; po_cur = po_nxt; m0_cur = m0_nxt; nb_cur = nb_nxt;
#pragma unroll
            for (int i = 0; i < 8; ++i) cur[i] = nxt[i];
        }
    }

    // ---- teardown
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc(tmem_base, TMEM_COLS);
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// tensor map of a row-major FP32 matrix [rows x cols] (cols contiguous, cols % 32 == 0): box = 32 cols x 256 rows, 128B swizzle
inline bool make_weight_map(CUtensorMap* map, const float* dptr, int rows, int cols) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)cols * sizeof(float)};
    cuuint32_t box[2] = {(cuuint32_t)TBK, (cuuint32_t)TBN};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(dptr), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

template <int MODE>
inline cudaError_t launch_chain_gemm_tc(const GemmArgs& g, const CUtensorMap& hi, const CUtensorMap& lo, int num_sms, cudaStream_t st) {
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(chain_gemm_tc_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const int tiles = (g.M / TBM) * ((g.N + TBN - 1) / TBN);
    const int grid = tiles < num_sms ? tiles : num_sms;
    chain_gemm_tc_kernel<MODE><<<grid, THREADS, SMEM_BYTES, st>>>(g, hi, lo);
    return cudaGetLastError();
}

}  // namespace tc
}  // namespace leb_nn

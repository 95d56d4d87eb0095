// nn_gemm_tc.cuh -- the CROWN chain contraction on the 5th-generation tensor cores (tcgen05), 3xTF32.
//
// One step of the back-substitution (eq. (18)) and one step of
// its reverse sweep are dense contractions  C[R x N] = T(A)[R x K] * W[K x N]  with
// R = tiles * rows (10^5 .. 10^6) coefficient rows, K, N = layer widths, W a weight matrix shared by
// all tiles.  FP32 operands are split  x = hi + lo  (hi = tf32(x), lo = tf32(x - hi)); the main term
// Whi*Ahi and the correction Whi*Alo + Wlo*Ahi are accumulated in FP32 in two separate tensor-memory
// accumulators and added in the epilogue (the tensor core truncates every accumulation, so the 2K/8
// correction MMAs must not touch the large accumulator).
//
// The product is computed TRANSPOSED, D[n, r] = sum_k W^T[n, k] T(A)[r, k]: the weights are the
// M-side operand (128 output columns per tile, TMA-staged), the coefficient rows the N-side operand
// (256 rows per tile).  A TMEM lane is then an output column: an epilogue thread owns one column,
// walks the rows, stores coalesced rows of C and -- in the reverse sweep -- keeps the column sums of
// the relaxation-parameter adjoints in registers (no cross-lane reduction).
//
// Kernel layout (persistent, one CTA per SM, 512 threads):
//   warp 0       TMA producer: pre-split weight tiles Whi, Wlo [128 x 32] (K-major, 128B swizzle)
//   warp 1       MMA issuer: 12 tcgen05.mma (M128 x N256 x K8) per 32-wide K slab
//   warp 2       TMEM allocation (512 columns: main [0,256), correction [256,512))
//   warp 3       forward: bulk-TMA loader of the K slab's per-neuron parameters
//   forward:       warps 4-7 epilogue (tcgen05.ld -> registers -> global), warps 8-15 row producers: global FP32 rows
//                  -> D = Lam^+ k_pos + Lam^- k_neg and the deviation-form constant gap += Lam^+ g_pos + Lam^- g_neg
//                  -> hi/lo split -> 128B-swizzled K-major shared-memory tiles (generic-proxy stores + async-proxy fence)
//   reverse sweep: warps 4-11 epilogue (two per TMEM lane quadrant, half of the tile's rows each), warps 12-15 row
//                  producers (plain rows, split only, 16 rows per thread)
// Stages are handed over with mbarriers: full[s] (producer arrivals + the TMA transaction), empty[s] (tcgen05.commit),
// tmem_full (tcgen05.commit), tmem_empty (epilogue arrivals).
// The forward step normally runs on CTA pairs instead (nn_gemm_tc2.cuh); this file's forward is LEB_FLAG_SINGLE_CTA.
#pragma once
#include <atomic>
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "nn_gemm_ffma.cuh"

namespace leb_nn {
namespace tc {

enum { MODE_FWD = 0, MODE_BWD = 1 };

constexpr int TBM = 128;      // output columns per tile (MMA M, weights)
constexpr int TBN = 256;      // coefficient rows per tile (MMA N)
constexpr int TBK = 32;
constexpr int WSTAGES = 3;    // weight ring (TMA: L2 latency ~ one K slab of MMA time, so one stage deeper than the rows)
constexpr int RSTAGES = 2;    // coefficient-row ring (register path, prefetched one slab ahead)
constexpr int W_TILE_BYTES = TBM * TBK * 4;                         // 16 KB (hi) + 16 KB (lo) per stage
constexpr int R_TILE_BYTES = TBN * TBK * 4;                         // 32 KB (hi) + 32 KB (lo) per stage
constexpr int RING_BYTES = WSTAGES * 2 * W_TILE_BYTES + RSTAGES * 2 * R_TILE_BYTES;   // 96 KB + 128 KB
constexpr int PSTAGES = 4;    // per-neuron parameter ring (tiny; four slabs ahead so that its latency never shows)
constexpr int PAR_BYTES = 5 * TBK * 4;                              // parameters of one K slab: kU, kL, phi', gU, gL
constexpr int BAR_BYTES = 192;
constexpr int SMEM_BYTES = RING_BYTES + PSTAGES * PAR_BYTES + BAR_BYTES;   // 226.7 KB of the 227 KB a CTA can have
constexpr int THREADS = 512;
constexpr int THREADS_BWD = 768;          // reverse sweep: 4 control + 16 epilogue + 4 producer warps
constexpr int PRODUCERS = 256;
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
// SLEEP_NS > 0: back off between probes (the roles that wait for a whole tile or slab must not take issue slots
// from the MMA warp that shares their scheduler)
template <int SLEEP_NS = 0>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    // try_wait suspends the thread for a hardware-defined time slice, so this is not a hot spin; the clock is only
    // consulted every 4096 slices to turn a protocol bug into a trap instead of a hung GPU
    uint32_t spins = 0;
    long long t0 = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (SLEEP_NS > 0) __nanosleep(SLEEP_NS);
        if ((++spins & 4095u) == 0u) {
            const long long now = clock64();
            if (t0 == 0) t0 = now;
            else if ((unsigned long long)(now - t0) > kSpinLimit) __trap();
        }
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
__device__ __forceinline__ void bulk_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
// hint: bring `bytes` (multiple of 16, 16-byte aligned) of global memory into L2
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
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
// NX consecutive FP32 columns of this warp's 32 TMEM lanes: thread t gets lane (warp%4)*32 + t, columns [c, c+NX).
// Asynchronous: tmem_ld_wait() before the registers are read.
template <int NX> __device__ __forceinline__ void tmem_ld(uint32_t taddr, float* v);
template <> __device__ __forceinline__ void tmem_ld<16>(uint32_t taddr, float* v) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
template <> __device__ __forceinline__ void tmem_ld<8>(uint32_t taddr, float* v) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
template <> __device__ __forceinline__ void tmem_ld<32>(uint32_t taddr, float* v) {
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
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// round to TF32 (10-bit mantissa), nearest with ties away from zero -- what cvt.rna.tf32.f32 computes for finite
// inputs, in two integer instructions (the PTX conversion expands to a longer NaN/Inf-aware sequence)
__device__ __forceinline__ float to_tf32(float x) {
    return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }

// register re-distribution between the warp roles (warpgroup granularity; 512 threads start with 128 registers each)
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

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


// per-tile geometry shared by the roles.  Tiles are numbered with the column block fastest, so the CTAs
// that run concurrently share coefficient rows (L2 reuse).  rows_pad % 256 == 0: a row block never
// straddles two trajectory tiles, so one slope-vector offset `po` serves the whole block.
struct TileGeo {
    int r0;        // first coefficient row of the block (global row index)
    int n0;        // first output column
    int rbase;     // r0 relative to its trajectory tile
    size_t po;     // offset of the tile's per-neuron parameter vectors
    bool rowsums;  // this column-block tile takes the row block's row sums (the gap)
};
__device__ __forceinline__ TileGeo tile_geo(const GemmArgs& g, int tile, int col_blocks) {
    TileGeo t;
    const int rb = tile / col_blocks;
    t.n0 = (tile - rb * col_blocks) * TBM;
    // a CTA's column block is fixed (grid % col_blocks == 0): rotate the tile that takes the row sums with the row block,
    // so that the extra work does not always land on the same CTAs
    t.rowsums = (tile - rb * col_blocks) == (rb % col_blocks);
    t.r0 = rb * TBN;
    const int tl = t.r0 / g.rows_pad;
    t.rbase = t.r0 - tl * g.rows_pad;
    t.po = (size_t)tl * g.ldp;
    return t;
}

// ---------------------------------------------------------------------------------------------
// reverse-sweep epilogue of one tile for one warp (shared by the single-CTA and the CTA-pair kernel): rows [c_lo, c_hi) of
// the tile's accumulator (TMEM address t_acc: this warp's lane quadrant, the tile's accumulator), output column n = lane.
// Masks the adjoint with the forward coefficients, writes C, keeps the five column sums in registers and
// adds them to the parameter adjoints.  release_acc() is called once, after the last TMEM read.
// ---------------------------------------------------------------------------------------------
template <int RB, int EPI_ROWS, class ReleaseFn>
__device__ __forceinline__ void bwd_epilogue_tile(const GemmArgs& g, int r0, int rbase, size_t po, int n, bool n_ok, int lane,
                                                  uint32_t t_acc, int c_lo, int c_hi, uint32_t tfull_bar, uint32_t acc_parity,
                                                  ReleaseFn release_acc) {
    // row kinds inside the block: [0,kb1) upper chain, [kb1,kb2) lower, [kb2,kbe) Jacobian, then padding
    const int kb1 = g.rows_kind - rbase, kb2 = 2 * g.rows_kind - rbase, kbe = g.nkinds * g.rows_kind - rbase;
    float kU = 0.f, kL = 0.f, gU = 0.f, gL = 0.f, dp = 0.f;
    if (n_ok) {
        kU = __ldg(g.kU + po + n); kL = __ldg(g.kL + po + n);
        gU = __ldg(g.gU + po + n); gL = __ldg(g.gL + po + n);
        dp = __ldg(g.dphi + po + n);
    }
    float skU = 0.f, skL = 0.f, sgU = 0.f, sgL = 0.f, sdb = 0.f;
    float* cbase = g.C + (size_t)r0 * g.ldc + n;
    const int kind0 = (0 >= kb1) + (0 >= kb2);
    const bool uniform = (kind0 == (TBN - 1 >= kb1) + (TBN - 1 >= kb2)) && (TBN - 1 < kbe) && (kind0 < 2);
    if (uniform) {
        // ---- all 256 rows on one chain (every hidden-layer target): no per-row selection
        const bool up = (kind0 == 0);
        const float kp = up ? kU : kL, kn = up ? kL : kU, gp = up ? gU : gL, gn = up ? gL : gU;
        const float* lp = g.Lam + (size_t)(g.lam_shared ? (rbase - kind0 * g.rows_kind) : r0) * g.ldl + (n_ok ? n : 0);
        // the gap adjoints of this warp's rows (EPI_ROWS <= 64): lane l holds rows c_lo + l and c_lo + 32 + l
        const float gbA = __ldg(g.gapbar + r0 + c_lo + lane);
        const float gbB = (EPI_ROWS > 32) ? __ldg(g.gapbar + r0 + c_lo + 32 + lane) : 0.f;
        auto ldr = [&](float* dst, int c) {
            const float* q = lp + (size_t)c * g.ldl;
#pragma unroll
            for (int j = 0; j < RB; ++j) dst[j] = __ldg(q + (size_t)j * g.ldl);
        };
        float sP = 0.f, sQ = 0.f, hP = 0.f, hQ = 0.f;
        // two coefficient buffers, 32 rows per loop trip: with 8 epilogue warps the 64-row / four-buffer version
        // spent 35-50 % of its samples on instruction-cache misses (stall_no_inst)
        float lam0[RB], lam1[RB];
        ldr(lam0, c_lo);
        mbar_wait<200>(tfull_bar, acc_parity);
        tc_fence_after();
        float a[RB];
        tmem_ld<RB>(t_acc + c_lo, a);
        float* cp = cbase + (size_t)c_lo * g.ldc;
        auto fstep = [&](int c, const float* P, float* L) {
            if (c + RB < c_hi) ldr(L, c + RB);
            const int rl = c - c_lo;                              // first row of the step inside the warp's range
            const float gbsrc = rl < 32 ? gbA : gbB;
            tmem_ld_wait();
            float d[RB];
#pragma unroll
            for (int j = 0; j < RB; ++j) d[j] = a[j];
            if (c + RB < c_hi) {
                tmem_ld<RB>(t_acc + c + RB, a);
            } else {                                         // last read of this accumulator: release it
                tc_fence_before();
                release_acc();
            }
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                const float gb = __shfl_sync(0xffffffffu, gbsrc, (rl & 31) + j);
                const float Db = d[j], lv = P[j];
                const float Pp = fmaxf(lv, 0.f), Q = fminf(lv, 0.f);
                sP = fmaf(Db, Pp, sP); sQ = fmaf(Db, Q, sQ);
                hP = fmaf(gb, Pp, hP); hQ = fmaf(gb, Q, hQ);
                const bool pos = lv > 0.f;
                float out = fmaf(Db, pos ? kp : kn, gb * (pos ? gp : gn));
                out = (lv == 0.f) ? 0.f : out;
                if (g.write_c && n_ok) *cp = out;
                cp += g.ldc;
            }
        };
#pragma unroll 1
        for (int c = c_lo; c < c_hi; c += 2 * RB) {
            fstep(c, lam0, lam1);
            fstep(c + RB, lam1, lam0);
        }
        skU = up ? sP : sQ; skL = up ? sQ : sP;
        sgU = up ? hP : hQ; sgL = up ? hQ : hP;
    } else {
        auto load_lam = [&](float* dst, int c) {
    #pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int jj = c + j;
                const int kind = (jj >= kb1) + (jj >= kb2);
                const int row = g.lam_shared ? (rbase + jj - kind * g.rows_kind) : (r0 + jj);
                dst[j] = (n_ok && jj < kbe) ? __ldg(g.Lam + (size_t)row * g.ldl + n) : 0.f;
            }
        };
        auto load_gb = [&](int c) {      // the rows' gap adjoints: lane j < 16 fetches row c + j, broadcast by shuffle
            const int jj = c + (lane & (RB - 1));
            const int kind = (jj >= kb1) + (jj >= kb2);
            return (jj < kbe && kind < 2) ? __ldg(g.gapbar + r0 + jj) : 0.f;
        };
        // forward coefficients one step (16 rows) ahead of their use -- they come from HBM; the first
        // steps are requested before the accumulator is complete and overlap the main loop
        float lam0[RB], lam1[RB];
        float gb0, gb1 = 0.f;
        load_lam(lam0, c_lo); gb0 = load_gb(c_lo);
        mbar_wait<200>(tfull_bar, acc_parity);
        tc_fence_after();
        float a[RB];
        tmem_ld<RB>(t_acc + c_lo, a);
        // one step: rows [c, c+16) with coefficients P / gap adjoints gbP; prefetch rows [c+16, c+32) into L
        auto estep = [&](int c, const float* P, float gbP, float* L, float& gbL) {
            if (c + RB < c_hi) { load_lam(L, c + RB); gbL = load_gb(c + RB); }
            tmem_ld_wait();
            float d[RB];
    #pragma unroll
            for (int j = 0; j < RB; ++j) d[j] = a[j];
            if (c + RB < c_hi) {
                tmem_ld<RB>(t_acc + c + RB, a);
            } else {                                             // last read of this accumulator: release it
                tc_fence_before();
                release_acc();
            }
    #pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int jj = c + j;
                const int kind = (jj >= kb1) + (jj >= kb2);            // warp-uniform
                const float gb = __shfl_sync(0xffffffffu, gbP, j);
                const float Db = d[j], lv = P[j];
                float out = 0.f;
                if (jj < kbe) {
                    if (kind == 2) {
                        sdb = fmaf(Db, lv, sdb);
                        out = Db * dp;
                    } else {
                        const bool up = (kind == 0);
                        const float Pp = fmaxf(lv, 0.f), Q = fminf(lv, 0.f);
                        const float dP = Db * Pp, dQ = Db * Q, gP = gb * Pp, gQ = gb * Q;
                        skU += up ? dP : dQ; skL += up ? dQ : dP;
                        sgU += up ? gP : gQ; sgL += up ? gQ : gP;
                        const float kp = up ? kU : kL, kn = up ? kL : kU, gp = up ? gU : gL, gn = up ? gL : gU;
                        out = lv > 0.f ? fmaf(Db, kp, gb * gp) : (lv < 0.f ? fmaf(Db, kn, gb * gn) : 0.f);
                    }
                }
                if (g.write_c && n_ok) cbase[(size_t)jj * g.ldc] = out;
            }
        };
    #pragma unroll 1
        for (int c = c_lo; c < c_hi; c += 2 * RB) {
            estep(c, lam0, gb0, lam1, gb1);
            estep(c + RB, lam1, gb1, lam0, gb0);
        }
    }
    if (n_ok) {
        atomicAdd(g.kUb + po + n, skU);
        atomicAdd(g.kLb + po + n, skL);
        atomicAdd(g.gUb + po + n, sgU);
        atomicAdd(g.gLb + po + n, sgL);
        if (g.nkinds == 3) atomicAdd(g.db + po + n, sdb);
    }
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(MODE == MODE_BWD ? THREADS_BWD : THREADS, 1)
chain_gemm_tc_kernel(const GemmArgs g, const __grid_constant__ CUtensorMap tm_hi, const __grid_constant__ CUtensorMap tm_lo) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t sbase = smem_u32(smem_raw);
    if ((sbase & 1023u) != 0u) __trap();                               // the 128B-swizzled tiles need 1024-byte alignment
    uint8_t* sgen = smem_raw;
    // weight ring: stage s = [Whi | Wlo]; row ring: stage s = [Rhi | Rlo]
    auto sW = [&](int s, int part) { return sbase + (2 * s + part) * W_TILE_BYTES; };
    auto sR = [&](int s, int part) { return sbase + WSTAGES * 2 * W_TILE_BYTES + (2 * s + part) * R_TILE_BYTES; };
    // parameter ring (forward only): stage s = [kU | kL | phi' | gU | gL] x 32 floats of one K slab
    auto sP = [&](int s) { return sbase + RING_BYTES + s * PAR_BYTES; };
    const uint32_t bar0 = sbase + RING_BYTES + PSTAGES * PAR_BYTES;
    auto bar_wfull = [&](int s) { return bar0 + 8 * s; };
    auto bar_wempty = [&](int s) { return bar0 + 8 * (WSTAGES + s); };
    auto bar_rfull = [&](int s) { return bar0 + 8 * (2 * WSTAGES + s); };
    auto bar_rempty = [&](int s) { return bar0 + 8 * (2 * WSTAGES + RSTAGES + s); };
    auto bar_tfull = [&](int a) { return bar0 + 8 * (2 * WSTAGES + 2 * RSTAGES + a); };
    auto bar_tempty = [&](int a) { return bar0 + 8 * (2 * WSTAGES + 2 * RSTAGES + 2 + a); };
    auto bar_pfull = [&](int s) { return bar0 + 8 * (2 * WSTAGES + 2 * RSTAGES + 4 + s); };
    auto bar_pempty = [&](int s) { return bar0 + 8 * (2 * WSTAGES + 2 * RSTAGES + 4 + PSTAGES + s); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sgen + RING_BYTES + PSTAGES * PAR_BYTES + 8 * (2 * WSTAGES + 2 * RSTAGES + 4 + 2 * PSTAGES));
    // forward: one accumulator pair (main [0,256), correction [256,512)); reverse sweep: the gradient tolerance
    // (1e-4) leaves room for the truncation of a single accumulator, so two of them alternate and the epilogue
    // of tile i overlaps the main loop of tile i+1
    constexpr int NACC = (MODE == MODE_BWD) ? 2 : 1;
    // Warp roles.  Forward: the row producers (transform + split) are the critical role: 4 epilogue warps (4..7), 8 producer
    // warps (8..15).  Reverse sweep: the producers only split, but the epilogue does ~35 instructions per row and one warp
    // per scheduler cannot issue them fast enough (ncu: producers 67 % idle, epilogue never): 768 threads -- 16 epilogue warps
    // (4..19, four per TMEM lane quadrant, each taking a quarter of the tile's 256 rows, 8 rows per step to fit 72 registers)
    // and 4 producer warps (20..23, 16 rows per thread).
    constexpr int kEpiWarps = (MODE == MODE_BWD) ? 16 : 4, kProdWarps = (MODE == MODE_BWD) ? 4 : 8;
    constexpr int kEpiRows = TBN * 4 / kEpiWarps;             // rows of the tile per epilogue warp

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int col_blocks = (g.N + TBM - 1) / TBM;
    const int row_blocks = g.M / TBN;                 // g.M % 256 == 0 (rows_pad % 256 == 0)
    const int num_tiles = row_blocks * col_blocks;
    const int nk = g.K / TBK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_hi);
        tma_prefetch_desc(&tm_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < WSTAGES; ++s) { mbar_init(bar_wfull(s), 1); mbar_init(bar_wempty(s), 1); }
        for (int s = 0; s < RSTAGES; ++s) { mbar_init(bar_rfull(s), kProdWarps * 32); mbar_init(bar_rempty(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(bar_tfull(a), 1); mbar_init(bar_tempty(a), kEpiWarps * 32); }
        for (int s = 0; s < PSTAGES; ++s) { mbar_init(bar_pfull(s), 1); mbar_init(bar_pempty(s), PRODUCERS / 32); }
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    // registers per thread: control warps 40; forward: epilogue 104, producers 184 (three slabs of rows in flight
    // plus the slopes of two); reverse sweep: epilogue 168 (four steps of forward coefficients in flight), producers 152
    // (the pool setmaxnreg redistributes is what the CTA got at launch: 512 x 128 registers forward, 768 x 80 = 61 440 in the
    // reverse sweep: 128 x 40 + 512 x 72 + 128 x 152 = 61 440)
    constexpr int kEpiRegs = (MODE == MODE_FWD) ? 104 : 72, kProdRegs = (MODE == MODE_FWD) ? 184 : 152;
    constexpr int RB = (MODE == MODE_BWD) ? 8 : 16;           // rows per step of the reverse-sweep epilogue

    if (warp < 4) reg_dec<40>();
    if (warp == 0) {
        // ===================== TMA producer (weights) =====================
        int stage = 0; uint32_t phase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            const TileGeo t = tile_geo(g, tile, col_blocks);
            const int n0 = t.n0;
            for (int kt = 0; kt < nk; ++kt) {
                mbar_wait<32>(bar_wempty(stage), phase ^ 1);
                if (lane == 0) {
                    mbar_arrive_expect_tx(bar_wfull(stage), 2 * W_TILE_BYTES);
                    tma_load_2d(sW(stage, 0), &tm_hi, kt * TBK, n0, bar_wfull(stage));
                    tma_load_2d(sW(stage, 1), &tm_lo, kt * TBK, n0, bar_wfull(stage));
                }
                __syncwarp();
                if (++stage == WSTAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 3) {
        // ===================== parameter loader (forward): the slab's slopes and gaps, four slabs ahead =====================
        if (MODE == MODE_FWD) {
            int stage = 0; uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                const TileGeo t = tile_geo(g, tile, col_blocks);
                for (int kt = 0; kt < nk; ++kt) {
                    mbar_wait<100>(bar_pempty(stage), phase ^ 1);
                    if (lane == 0) {
                        const size_t o = t.po + (size_t)kt * TBK;
                        mbar_arrive_expect_tx(bar_pfull(stage), PAR_BYTES);
                        bulk_load_1d(sP(stage) + 0 * TBK * 4, g.kU + o, TBK * 4, bar_pfull(stage));
                        bulk_load_1d(sP(stage) + 1 * TBK * 4, g.kL + o, TBK * 4, bar_pfull(stage));
                        bulk_load_1d(sP(stage) + 2 * TBK * 4, g.dphi + o, TBK * 4, bar_pfull(stage));
                        bulk_load_1d(sP(stage) + 3 * TBK * 4, g.gU + o, TBK * 4, bar_pfull(stage));
                        bulk_load_1d(sP(stage) + 4 * TBK * 4, g.gL + o, TBK * 4, bar_pfull(stage));
                    }
                    __syncwarp();
                    if (++stage == PSTAGES) { stage = 0; phase ^= 1; }
                }
            }
        } else if (!g.lam_shared) {
            // ===================== reverse sweep: L2 prefetch of the forward coefficients the epilogue will read =====================
            // The epilogue reads its tile's 256 x 128 block of Lambda_l from HBM with short register prefetch (ncu: half of its
            // samples wait on those loads).  When the accumulator of tile i becomes free -- i.e. as its main loop starts -- this
            // warp asks for the block to be brought into L2 (512 B per row), a whole main loop ahead of the epilogue.
            int tcount = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcount) {
                const int acc = tcount % NACC;
                const uint32_t par = (uint32_t)(((tcount / NACC) & 1) ^ 1);
                for (int probe = 0; probe < 200000 && !mbar_try_wait(bar_tempty(acc), par); ++probe) __nanosleep(100);   // a hint: never block
                const TileGeo t = tile_geo(g, tile, col_blocks);
                const int cols = (g.N - t.n0) < TBM ? (g.N - t.n0) : TBM;
                const float* base = g.Lam + (size_t)t.r0 * g.ldl + t.n0;
                for (int j = lane; j < TBN; j += 32) bulk_prefetch_l2(base + (size_t)j * g.ldl, (uint32_t)cols * 4u);
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        int ws = 0, rs = 0; uint32_t wphase = 0, rphase = 0;
        const uint32_t idesc = make_idesc(TBM, TBN);
        const uint64_t dW0 = make_smem_desc(sW(0, 0)), dR0 = make_smem_desc(sR(0, 0));   // stage 0, hi part; the others are offsets
        int tcount = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcount) {
            const int acc = tcount % NACC;
            mbar_wait(bar_tempty(acc), ((tcount / NACC) & 1) ^ 1);          // the epilogue has drained this accumulator
            tc_fence_after();
            const uint32_t d_main = tmem_base + acc * TBN;
            const uint32_t d_corr = (MODE == MODE_BWD) ? d_main : tmem_base + TBN;
            for (int kt = 0; kt < nk; ++kt) {
                mbar_wait(bar_wfull(ws), wphase);
                mbar_wait(bar_rfull(rs), rphase);
                tc_fence_after();
                // warp-uniform descriptor arithmetic stays outside the single-lane region (uniform datapath)
                const uint64_t whi = dW0 + (uint64_t)((2 * ws * W_TILE_BYTES) >> 4), wlo = whi + (W_TILE_BYTES >> 4);
                const uint64_t rhi = dR0 + (uint64_t)((2 * rs * R_TILE_BYTES) >> 4), rlo = rhi + (R_TILE_BYTES >> 4);
                if (lane == 0) {
#pragma unroll
                    for (int k = 0; k < TBK / 8; ++k) {
                        const uint64_t ko = (uint64_t)(k * 32 >> 4);     // 8 tf32 = 32 bytes along K inside the swizzle atom
                        if (MODE == MODE_BWD) {
                            umma_tf32(d_main, whi + ko, rlo + ko, idesc, (kt | k) != 0);
                            umma_tf32(d_main, wlo + ko, rhi + ko, idesc, 1u);
                            umma_tf32(d_main, whi + ko, rhi + ko, idesc, 1u);
                        } else {
                            umma_tf32(d_main, whi + ko, rhi + ko, idesc, (kt | k) != 0);
                            umma_tf32(d_corr, whi + ko, rlo + ko, idesc, (kt | k) != 0);
                            umma_tf32(d_corr, wlo + ko, rhi + ko, idesc, 1u);
                        }
                    }
                    umma_commit(bar_wempty(ws));                         // both stages are free when these MMAs retire
                    umma_commit(bar_rempty(rs));
                    if (kt == nk - 1) umma_commit(bar_tfull(acc));       // accumulators complete
                }
                __syncwarp();
                if (++ws == WSTAGES) { ws = 0; wphase ^= 1; }
                if (++rs == RSTAGES) { rs = 0; rphase ^= 1; }
            }
        }
    } else if (warp >= 4 && warp < 4 + kEpiWarps) {
        // ===================== epilogue: TMEM lane = output column, TMEM column = coefficient row =====================
        if (kEpiRegs < 128) reg_dec<kEpiRegs>(); else reg_inc<kEpiRegs>();
        const int q = (MODE == MODE_BWD) ? (warp & 3) : (warp - 4);          // TMEM lane quadrant of this warp (warp % 4)
        const int c_lo = (MODE == MODE_BWD) ? ((warp - 4) >> 2) * kEpiRows : 0, c_hi = c_lo + kEpiRows;   // this warp's rows of the tile
        const uint32_t t_lane = tmem_base + ((uint32_t)(q * 32) << 16);
        int tcount = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcount) {
            const TileGeo t = tile_geo(g, tile, col_blocks);
            const int n = t.n0 + q * 32 + lane;                  // this thread's output column
            const bool n_ok = n < g.N;
            const int acc = tcount % NACC;
            const uint32_t acc_parity = (tcount / NACC) & 1;
            if (MODE == MODE_FWD) {
                mbar_wait<200>(bar_tfull(acc), acc_parity);
                tc_fence_after();
                float* cbase = g.C + (size_t)t.r0 * g.ldc + n;
                // 16 rows per step, the TMEM loads of step i+1 in flight while step i is stored
                float a0[16], b0[16], a1[16], b1[16];
                tmem_ld<16>(t_lane, a0);
                tmem_ld<16>(t_lane + TBN, b0);
#pragma unroll 1
                for (int c = 0; c < TBN; c += 32) {
                    tmem_ld_wait();
                    tmem_ld<16>(t_lane + c + 16, a1);
                    tmem_ld<16>(t_lane + TBN + c + 16, b1);
                    if (n_ok) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) cbase[(size_t)(c + j) * g.ldc] = a0[j] + b0[j];   // 128 B per warp and row
                    }
                    tmem_ld_wait();
                    if (c + 32 < TBN) {
                        tmem_ld<16>(t_lane + c + 32, a0);
                        tmem_ld<16>(t_lane + TBN + c + 32, b0);
                    } else {                                             // last read of this tile's accumulators: release them
                        tc_fence_before();
                        mbar_arrive(bar_tempty(acc));
                    }
                    if (n_ok) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) cbase[(size_t)(c + 16 + j) * g.ldc] = a1[j] + b1[j];
                    }
                }
            } else {
                bwd_epilogue_tile<RB, kEpiRows>(g, t.r0, t.rbase, t.po, n, n_ok, lane, t_lane + acc * TBN, c_lo, c_hi, bar_tfull(acc),
                                                acc_parity, [&]() { mbar_arrive(bar_tempty(acc)); });
            }
        }
    } else if (MODE == MODE_BWD && warp >= 4 + kEpiWarps) {
        // ===================== row producers, reverse sweep: plain rows, hi/lo split only =====================
        // 4 warps; warp pw owns rows [pw*64, pw*64 + 64) of the block, a thread 16 of them (8 threads per row, one float4
        // each).  Two register buffers: the loads of slab i+1 are in flight while slab i is split and stored.
        reg_inc<kProdRegs>();
        const int pw = warp - (4 + kEpiWarps);
        const int r4 = lane >> 3, c4 = lane & 7;
        const float4* const A4 = reinterpret_cast<const float4*>(g.A);
        const uint32_t rstride = (uint32_t)(g.lda >> 2) * 4u;          // 4 rows, in float4 units
        int ltile = blockIdx.x, lkt = 0;
        bool lhave = ltile < num_tiles;
        uint32_t lbase = 0;
        auto set_base = [&]() { lbase = (uint32_t)(((size_t)(ltile / col_blocks * TBN + pw * 64 + r4) * g.lda) >> 2) + c4; };
        auto issue = [&](float4* buf) {
            if (!lhave) return;
            const float4* src = A4 + lbase + (uint32_t)lkt * (TBK / 4);
#pragma unroll
            for (int i = 0; i < 16; ++i) buf[i] = __ldg(src + (size_t)i * rstride);
            if (++lkt == nk) {
                lkt = 0;
                ltile += gridDim.x;
                lhave = ltile < num_tiles;
                if (lhave) set_base();
            }
        };
        int stage = 0; uint32_t phase = 0;
        int remaining = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) remaining += nk;
        auto put = [&](const float4* buf) {
            mbar_wait(bar_rempty(stage), phase ^ 1);
            const uint32_t r_hi = sR(stage, 0), r_lo = sR(stage, 1);
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                const float4 v = buf[i];
                float4 hi, lo;
                hi.x = to_tf32(v.x); hi.y = to_tf32(v.y); hi.z = to_tf32(v.z); hi.w = to_tf32(v.w);
                lo.x = v.x - hi.x; lo.y = v.y - hi.y; lo.z = v.z - hi.z; lo.w = v.w - hi.w;
                const int row = pw * 64 + i * 4 + r4;
                const uint32_t off = (uint32_t)row * 128u + (uint32_t)((c4 ^ (row & 7)) << 4);     // 128B swizzle
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(r_hi + off), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w) : "memory");
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(r_lo + off), "f"(lo.x), "f"(lo.y), "f"(lo.z), "f"(lo.w) : "memory");
            }
            fence_proxy_async();
            mbar_arrive(bar_rfull(stage));
            if (++stage == RSTAGES) { stage = 0; phase ^= 1; }
        };
        if (lhave) {
            float4 b0[16], b1[16];
            set_base();
            issue(b0);
            while (true) {
                issue(b1);
                put(b0);
                if (--remaining == 0) break;
                issue(b0);
                put(b1);
                if (--remaining == 0) break;
            }
        }
    } else if (MODE == MODE_FWD && warp >= 8) {
        // ===================== row producers =====================
        // Two cursors walk the CTA's sequence of (tile, K slab): the LOADER issues the global loads of a slab
        // into one of three register buffers two slabs ahead of the TRANSFORMER, which relaxes, splits and
        // stores the oldest buffer into the stage the MMA warp has released.  HBM latency (~1.5 slabs of MMA
        // time) is covered by the two slabs in flight; the per-neuron slopes are fetched one slab ahead.
        reg_inc<kProdRegs>();
        const int pw = warp - 8;                   // 0..7: this warp owns rows [pw*32, pw*32 + 32) of the block
        const int r4 = lane >> 3, c4 = lane & 7;   // 8 threads per row (one float4 each = 128 B), 4 rows per warp instruction
        const float4* const A4 = reinterpret_cast<const float4*>(g.A);
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        // ---- loader cursor
        int ltile = blockIdx.x, lkt = 0;
        bool lhave = ltile < num_tiles;
        uint32_t aoff[8];                          // row offsets into A in float4 units
        uint32_t lkinds = 0;                       // 2 bits per row: 0 upper, 1 lower, 2 Jacobian chain, 3 padding
        auto setup_load = [&]() {
            const TileGeo t = tile_geo(g, ltile, col_blocks);
            lkinds = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int j = pw * 32 + i * 4 + r4;
                if (MODE == MODE_FWD) {
                    const int rin = t.rbase + j;
                    int kind = rin / g.rows_kind;
                    int rk = rin - kind * g.rows_kind;
                    if (kind >= g.nkinds) { kind = 3; rk = 0; }
                    aoff[i] = (uint32_t)(((size_t)(g.a_shared ? rk : (t.r0 + j)) * g.lda) >> 2) + c4;
                    lkinds |= (uint32_t)kind << (2 * i);
                } else {
                    aoff[i] = (uint32_t)(((size_t)(t.r0 + j) * g.lda) >> 2) + c4;
                }
            }
        };
        auto issue = [&](float4* buf, uint32_t& bkinds) {
            bkinds = lkinds;
            if (!lhave) return;
            const uint32_t ko = (uint32_t)lkt * (TBK / 4);
            if ((lkinds & (lkinds >> 1) & 0x5555u) == 0u) {          // no padding row among this thread's eight
#pragma unroll
                for (int i = 0; i < 8; ++i) buf[i] = __ldg(A4 + aoff[i] + ko);
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const bool ok = ((lkinds >> (2 * i)) & 3u) != 3u;
                    buf[i] = ok ? __ldg(A4 + aoff[i] + ko) : zero4;
                }
            }
            if (++lkt == nk) {
                lkt = 0;
                ltile += gridDim.x;
                lhave = ltile < num_tiles;
                if (lhave) setup_load();
            }
        };
        // ---- transformer cursor
        int ptile = blockIdx.x, pkt = 0;
        bool phave = ptile < num_tiles;
        TileGeo t_cur = tile_geo(g, phave ? ptile : 0, col_blocks);
        int stage = 0; uint32_t phase = 0;
        int ps = 0; uint32_t pphase = 0;           // parameter stage of the slab being transformed
        auto lds4 = [&](uint32_t addr) {
            float4 v;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
            return v;
        };
        auto split_store = [&](const float4& v, uint32_t r_hi, uint32_t r_lo, int row) {
            // hi = tf32(v) (nearest); lo = v - hi exactly (|lo| <= 2^-11 |v|, at most 13 significant bits); the tensor
            // core reads the upper 19 bits of lo, i.e. lo to within 2^-10 |lo| <= 2^-21 |v|
            float4 hi, lo;
            hi.x = to_tf32(v.x); hi.y = to_tf32(v.y); hi.z = to_tf32(v.z); hi.w = to_tf32(v.w);
            lo.x = v.x - hi.x; lo.y = v.y - hi.y; lo.z = v.z - hi.z; lo.w = v.w - hi.w;
            const uint32_t off = (uint32_t)row * 128u + (uint32_t)((c4 ^ (row & 7)) << 4);     // 128B swizzle
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(r_hi + off), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w) : "memory");
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(r_lo + off), "f"(lo.x), "f"(lo.y), "f"(lo.z), "f"(lo.w) : "memory");
        };
        auto relax4 = [&](float4& v, const float4& kp, const float4& kn) {
            v.x *= v.x > 0.f ? kp.x : kn.x;
            v.y *= v.y > 0.f ? kp.y : kn.y;
            v.z *= v.z > 0.f ? kp.z : kn.z;
            v.w *= v.w > 0.f ? kp.w : kn.w;
        };
        auto gap4 = [&](const float4& v, const float4& gp, const float4& gn) {
            return (v.x > 0.f ? v.x * gp.x : v.x * gn.x) + (v.y > 0.f ? v.y * gp.y : v.y * gn.y) +
                   (v.z > 0.f ? v.z * gp.z : v.z * gn.z) + (v.w > 0.f ? v.w * gp.w : v.w * gn.w);
        };
        float gsum[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) gsum[i] = 0.f;

        // one step: prefetch into L (two slabs ahead), transform P (kinds kP); returns false after the last slab
        auto step = [&](float4* P, uint32_t kP, float4* L, uint32_t& kL) -> bool {
            issue(L, kL);
            // position of the next slab to transform
            int ntile = ptile, nkt = pkt + 1;
            TileGeo t_nxt = t_cur;
            if (nkt == nk) { nkt = 0; ntile = ptile + gridDim.x; }
            const bool nhave = ntile < num_tiles;
            if (nhave && nkt == 0) t_nxt = tile_geo(g, ntile, col_blocks);
            const bool do_gap = (MODE == MODE_FWD) && t_cur.rowsums && (g.gap != nullptr);
            float4 kUc = zero4, kLc = zero4, dpc = zero4, gU4 = zero4, gL4 = zero4;
            int p_used = 0;
            if (MODE == MODE_FWD) {
                mbar_wait(bar_pfull(ps), pphase);
                const uint32_t pp = sP(ps) + c4 * 16;
                kUc = lds4(pp); kLc = lds4(pp + TBK * 4);
                if (g.nkinds == 3) dpc = lds4(pp + 2 * TBK * 4);
                if (do_gap) { gU4 = lds4(pp + 3 * TBK * 4); gL4 = lds4(pp + 4 * TBK * 4); }
                // the loads must have returned before the stage is handed back to the async proxy
                p_used = ps;                                             // released below, behind the step's proxy fence
                if (++ps == PSTAGES) { ps = 0; pphase ^= 1; }
            }
            mbar_wait(bar_rempty(stage), phase ^ 1);
            const uint32_t r_hi = sR(stage, 0), r_lo = sR(stage, 1);
            if (MODE == MODE_FWD && (kP == 0u || kP == 0x5555u)) {
                // all 8 rows of this thread on one chain (always the case for hidden-layer targets)
                const float4 kp = kP == 0u ? kUc : kLc, kn = kP == 0u ? kLc : kUc;
                const float4 gp = kP == 0u ? gU4 : gL4, gn = kP == 0u ? gL4 : gU4;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    float4 v = P[i];
                    if (do_gap) gsum[i] += gap4(v, gp, gn);
                    relax4(v, kp, kn);
                    split_store(v, r_hi, r_lo, pw * 32 + i * 4 + r4);
                }
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    float4 v = P[i];
                    if (MODE == MODE_FWD) {
                        const uint32_t kind = (kP >> (2 * i)) & 3u;
                        if (kind < 2u) {
                            if (do_gap) gsum[i] += gap4(v, kind == 0u ? gU4 : gL4, kind == 0u ? gL4 : gU4);
                            relax4(v, kind == 0u ? kUc : kLc, kind == 0u ? kLc : kUc);
                        } else if (kind == 2u) {
                            relax4(v, dpc, dpc);
                        }
                    }
                    split_store(v, r_hi, r_lo, pw * 32 + i * 4 + r4);
                }
            }
            // one cross-proxy fence for both hand-overs: the row stores become visible to the tensor core, and the
            // parameter reads above are ordered before the bulk TMA that recycles their stage (without a fence on that
            // path ~10 % of config-5 tiles came out wrong, non-deterministically)
            fence_proxy_async();
            mbar_arrive(bar_rfull(stage));
            if (++stage == RSTAGES) { stage = 0; phase ^= 1; }
            if (MODE == MODE_FWD) {
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_pempty(p_used));
            }
            // ---- end of a tile: the deviation-form constant (row sums over K; 8 threads per row)
            if (pkt == nk - 1) {
                if (do_gap) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        float s = gsum[i];
                        s += __shfl_xor_sync(0xffffffffu, s, 1);
                        s += __shfl_xor_sync(0xffffffffu, s, 2);
                        s += __shfl_xor_sync(0xffffffffu, s, 4);
                        const int m = t_cur.r0 + pw * 32 + i * 4 + r4;
                        if (c4 == 0) g.gap[m] = (g.gap_init ? 0.f : g.gap[m]) + s;
                    }
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) gsum[i] = 0.f;
            }
            ptile = ntile; pkt = nkt; t_cur = t_nxt;
            return nhave;
        };
        if (phave) {
            float4 b0[8], b1[8], b2[8];
            uint32_t k0 = 0, k1 = 0, k2 = 0;
            setup_load();
            issue(b0, k0);
            issue(b1, k1);
            while (true) {
                if (!step(b0, k0, b2, k2)) break;
                if (!step(b1, k1, b0, k0)) break;
                if (!step(b2, k2, b1, k1)) break;
            }
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

// tensor map of a row-major FP32 matrix [rows x cols] (cols contiguous, cols % 32 == 0): box = 32 cols x 128 rows,
// 128B swizzle; rows beyond the matrix are zero-filled
inline bool make_weight_map(CUtensorMap* map, const float* dptr, int rows, int cols) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)cols * sizeof(float)};
    cuuint32_t box[2] = {(cuuint32_t)TBK, (cuuint32_t)TBM};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(dptr), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// g.M (coefficient rows) must be a multiple of 256, g.K and g.N multiples of 32
template <int MODE>
inline cudaError_t launch_chain_gemm_tc(const GemmArgs& g, const CUtensorMap& hi, const CUtensorMap& lo, int num_sms, cudaStream_t st) {
    // the attribute is per device: one bit per device ordinal (a context may live on any GPU of the process)
    static std::atomic<unsigned long long> attr_done{0ull};
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned long long bit = 1ull << (dev & 63);
    if (!(attr_done.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(chain_gemm_tc_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return e;
        attr_done.fetch_or(bit, std::memory_order_release);
    }
    if (g.M % TBN != 0 || g.K % TBK != 0) return cudaErrorInvalidValue;
    const int tiles = (g.M / TBN) * ((g.N + TBM - 1) / TBM);
    const int grid = tiles < num_sms ? tiles : num_sms;
    chain_gemm_tc_kernel<MODE><<<grid, MODE == MODE_BWD ? THREADS_BWD : THREADS, SMEM_BYTES, st>>>(g, hi, lo);
    return cudaGetLastError();
}

}  // namespace tc
}  // namespace leb_nn

// nn_gemm_tc2.cuh -- forward CROWN chain step (eq. (18)) on CTA PAIRS: tcgen05.mma.cta_group::2.
//
// Same contraction, operands, 3xTF32 split and two-accumulator scheme as nn_gemm_tc.cuh (read that header first).
// What changes: the forward kernel is bound by its row producers (global FP32 row -> relax -> hi/lo split -> swizzled
// st.shared; ncu: 90 % busy while the tensor pipe is 50 % active).  A pair of CTAs (cluster of 2, one TPC) computes a
// 256-column x 256-row tile with M = 256 MMAs issued by the leader: each CTA stages only ITS 128 weight rows (A operand,
// its own output columns) and transforms only ITS 128 coefficient rows (B operand, N/2 each).  Per SM the producer work
// and the row traffic from L2 halve; the tensor work per SM is unchanged.  The row ring gets 4 stages of 32 KB.
//
// The waits are plain CTA-scope mbarrier waits: what crosses the CTA boundary is read by the tensor core (async proxy) out
// of shared memory, never by generic loads, so no cluster-scope acquire (an L1 invalidate per probe: 21 % of the kernel's
// samples when it was there) is needed; the writers fence their own shared memory for the async proxy and release at
// cluster scope.
//
// Cross-CTA protocol (all barriers sit at the same shared-memory offsets in both CTAs):
//   wfull[s], rfull[s], tempty   live in the LEADER (rank 0): the peer's TMA completes its bytes on the leader's wfull
//                                (cp.async.bulk.tensor ... .cta_group::2), the peer's producers / epilogue threads arrive
//                                remotely (mapa + mbarrier.arrive.shared::cluster; a cluster-scope
//                                release there waits for the producers' own prefetch loads: 12 % of their samples)
//   wempty[s], rempty[s], tfull  exist in BOTH CTAs and are signalled together by the leader's
//                                tcgen05.commit.cta_group::2 ... .multicast::cluster (mask 0b11)
#pragma once
#include <atomic>
#include "nn_gemm_tc.cuh"

namespace leb_nn {
namespace tc2 {

using namespace tc;

constexpr int HROWS = TBN / 2;                                   // coefficient rows a CTA transforms per tile
constexpr int R2STAGES = 4;
constexpr int R2_TILE_BYTES = HROWS * TBK * 4;                   // 16 KB (hi) + 16 KB (lo) per stage
constexpr int RING2_BYTES = WSTAGES * 2 * W_TILE_BYTES + R2STAGES * 2 * R2_TILE_BYTES;   // 96 KB + 128 KB
constexpr int SMEM2_BYTES = RING2_BYTES + PSTAGES * PAR_BYTES + 256;

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the barrier at the same offset in CTA `rank` of the cluster
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar, uint32_t rank) {
    asm volatile(
        "{\n"
        ".reg .b32 ra;\n"
        "mapa.shared::cluster.u32 ra, %0, %1;\n"
        "mbarrier.arrive.shared::cluster.b64 _, [ra];\n"
        "}\n" ::"r"(bar), "r"(rank)
        : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cluster(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
    uint32_t spins = 0;
    long long t0 = 0;
    while (!mbar_try_wait_cluster(bar, parity)) {
        if ((++spins & 4095u) == 0u) {
            const long long now = clock64();
            if (t0 == 0) t0 = now;
            else if ((unsigned long long)(now - t0) > kSpinLimit) __trap();
        }
    }
}
// TMA tile load whose completion bytes go to the barrier at the same offset in the pair's leader CTA
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    const uint32_t lbar = bar & 0xFEFFFFFFu;                     // clear the CTA-rank bit: the leader's copy of the barrier
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(lbar)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc_pair(uint32_t dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void umma_tf32_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// arrive (once the MMAs issued so far have retired) on the barrier at this offset in BOTH CTAs of the pair
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(bar), "h"((uint16_t)3)
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

struct PairGeo {
    int r0;        // first coefficient row of the 256-row block
    int n0;        // first output column of THIS CTA (pair column block * 256 + rank * 128)
    int rbase;     // r0 relative to its trajectory tile
    size_t po;     // offset of the tile's per-neuron parameter vectors
    bool rowsums;  // this pair tile takes the row block's row sums (the gap)
};
__device__ __forceinline__ PairGeo pair_geo(const GemmArgs& g, int ptile, int col_pairs, int rank) {
    PairGeo t;
    const int rb = ptile / col_pairs, cp = ptile - rb * col_pairs;
    t.n0 = cp * 2 * TBM + rank * TBM;
    t.rowsums = cp == (rb % col_pairs);
    t.r0 = rb * TBN;
    const int tl = t.r0 / g.rows_pad;
    t.rbase = t.r0 - tl * g.rows_pad;
    t.po = (size_t)tl * g.ldp;
    return t;
}

// ---------------------------------------------------------------------------------------------
// the kernel (forward chain step only; the reverse sweep is epilogue-bound and stays on single CTAs)
// ---------------------------------------------------------------------------------------------
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
chain_gemm_tc2_fwd_kernel(const GemmArgs g, const __grid_constant__ CUtensorMap tm_hi, const __grid_constant__ CUtensorMap tm_lo) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t sbase = smem_u32(smem_raw);
    if ((sbase & 1023u) != 0u) __trap();
    uint8_t* sgen = smem_raw;
    auto sW = [&](int s, int part) { return sbase + (2 * s + part) * W_TILE_BYTES; };
    auto sR = [&](int s, int part) { return sbase + WSTAGES * 2 * W_TILE_BYTES + (2 * s + part) * R2_TILE_BYTES; };
    auto sP = [&](int s) { return sbase + RING2_BYTES + s * PAR_BYTES; };
    const uint32_t bar0 = sbase + RING2_BYTES + PSTAGES * PAR_BYTES;
    auto bar_wfull = [&](int s) { return bar0 + 8 * s; };
    auto bar_wempty = [&](int s) { return bar0 + 8 * (WSTAGES + s); };
    auto bar_rfull = [&](int s) { return bar0 + 8 * (2 * WSTAGES + s); };
    auto bar_rempty = [&](int s) { return bar0 + 8 * (2 * WSTAGES + R2STAGES + s); };
    const uint32_t bar_tfull = bar0 + 8 * (2 * WSTAGES + 2 * R2STAGES);
    const uint32_t bar_tempty = bar_tfull + 8;
    auto bar_pfull = [&](int s) { return bar_tfull + 16 + 8 * s; };
    auto bar_pempty = [&](int s) { return bar_tfull + 16 + 8 * (PSTAGES + s); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sgen + RING2_BYTES + PSTAGES * PAR_BYTES + 8 * (2 * WSTAGES + 2 * R2STAGES + 2 + 2 * PSTAGES));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const bool leader = rank == 0;
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
    const int col_pairs = (g.N + 2 * TBM - 1) / (2 * TBM);
    const int row_blocks = g.M / TBN;
    const int num_tiles = row_blocks * col_pairs;
    const int nk = g.K / TBK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_hi);
        tma_prefetch_desc(&tm_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < WSTAGES; ++s) { mbar_init(bar_wfull(s), 1); mbar_init(bar_wempty(s), 1); }
        for (int s = 0; s < R2STAGES; ++s) { mbar_init(bar_rfull(s), 2 * PRODUCERS / 32); mbar_init(bar_rempty(s), 1); }
        mbar_init(bar_tfull, 1);
        mbar_init(bar_tempty, 2 * 4);
        for (int s = 0; s < PSTAGES; ++s) { mbar_init(bar_pfull(s), 1); mbar_init(bar_pempty(s), PRODUCERS / 32); }
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc_pair(smem_u32(tmem_slot), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                                   // both CTAs' barriers exist before any remote arrive / multicast commit
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp < 4) reg_dec<40>();
    if (warp == 0) {
        // ===================== TMA producer: this CTA's 128 weight rows; bytes complete on the leader's barrier =====================
        int stage = 0; uint32_t phase = 0;
        for (int tile = pair; tile < num_tiles; tile += npairs) {
            const PairGeo t = pair_geo(g, tile, col_pairs, (int)rank);
            for (int kt = 0; kt < nk; ++kt) {
                mbar_wait<32>(bar_wempty(stage), phase ^ 1);
                if (lane == 0) {
                    if (leader) mbar_arrive_expect_tx(bar_wfull(stage), 4 * W_TILE_BYTES);     // both CTAs' hi + lo tiles
                    tma_load_2d_pair(sW(stage, 0), &tm_hi, kt * TBK, t.n0, bar_wfull(stage));
                    tma_load_2d_pair(sW(stage, 1), &tm_lo, kt * TBK, t.n0, bar_wfull(stage));
                }
                __syncwarp();
                if (++stage == WSTAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 3) {
        // ===================== parameter loader (local to each CTA) =====================
        int stage = 0; uint32_t phase = 0;
        for (int tile = pair; tile < num_tiles; tile += npairs) {
            const PairGeo t = pair_geo(g, tile, col_pairs, (int)rank);
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
    } else if (warp == 1) {
        // ===================== MMA issuer: the leader only, M = 256 (128 output columns per CTA) x N = 256 (128 rows per CTA) =====================
        if (leader) {
            int ws = 0, rs = 0; uint32_t wphase = 0, rphase = 0;
            const uint32_t idesc = make_idesc(2 * TBM, TBN);
            const uint64_t dW0 = make_smem_desc(sW(0, 0)), dR0 = make_smem_desc(sR(0, 0));
            const uint32_t d_main = tmem_base, d_corr = tmem_base + TBN;
            int tcount = 0;
            for (int tile = pair; tile < num_tiles; tile += npairs, ++tcount) {
                mbar_wait(bar_tempty, (tcount & 1) ^ 1);                 // both CTAs' epilogues have drained the accumulators
                tc_fence_after();
                for (int kt = 0; kt < nk; ++kt) {
                    mbar_wait(bar_wfull(ws), wphase);
                    mbar_wait(bar_rfull(rs), rphase);
                    tc_fence_after();
                    const uint64_t whi = dW0 + (uint64_t)((2 * ws * W_TILE_BYTES) >> 4), wlo = whi + (W_TILE_BYTES >> 4);
                    const uint64_t rhi = dR0 + (uint64_t)((2 * rs * R2_TILE_BYTES) >> 4), rlo = rhi + (R2_TILE_BYTES >> 4);
                    if (lane == 0) {
#pragma unroll
                        for (int k = 0; k < TBK / 8; ++k) {
                            const uint64_t ko = (uint64_t)(k * 32 >> 4);
                            umma_tf32_pair(d_main, whi + ko, rhi + ko, idesc, (kt | k) != 0);
                            umma_tf32_pair(d_corr, whi + ko, rlo + ko, idesc, (kt | k) != 0);
                            umma_tf32_pair(d_corr, wlo + ko, rhi + ko, idesc, 1u);
                        }
                        umma_commit_pair(bar_wempty(ws));
                        umma_commit_pair(bar_rempty(rs));
                        if (kt == nk - 1) umma_commit_pair(bar_tfull);
                    }
                    __syncwarp();
                    if (++ws == WSTAGES) { ws = 0; wphase ^= 1; }
                    if (++rs == R2STAGES) { rs = 0; rphase ^= 1; }
                }
            }
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== epilogue: this CTA's 128 output columns (TMEM lanes) x all 256 rows =====================
        reg_dec<104>();
        const int q = warp - 4;
        const uint32_t t_lane = tmem_base + ((uint32_t)(q * 32) << 16);
        int tcount = 0;
        for (int tile = pair; tile < num_tiles; tile += npairs, ++tcount) {
            const PairGeo t = pair_geo(g, tile, col_pairs, (int)rank);
            const int n = t.n0 + q * 32 + lane;
            const bool n_ok = n < g.N;
            mbar_wait<200>(bar_tfull, tcount & 1);
            tc_fence_after();
            float* cbase = g.C + (size_t)t.r0 * g.ldc + n;
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
                    for (int j = 0; j < 16; ++j) cbase[(size_t)(c + j) * g.ldc] = a0[j] + b0[j];
                }
                tmem_ld_wait();
                if (c + 32 < TBN) {
                    tmem_ld<16>(t_lane + c + 32, a0);
                    tmem_ld<16>(t_lane + TBN + c + 32, b0);
                } else {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) { if (leader) mbar_arrive(bar_tempty); else mbar_arrive_remote(bar_tempty, 0); }
                }
                if (n_ok) {
#pragma unroll
                    for (int j = 0; j < 16; ++j) cbase[(size_t)(c + 16 + j) * g.ldc] = a1[j] + b1[j];
                }
            }
        }
    } else if (warp >= 8) {
        // ===================== row producers: this CTA's 128 rows of the block, 4 rows per thread =====================
        reg_inc<184>();
        const int pw = warp - 8;                   // warp pw owns local rows [pw*16, pw*16 + 16)
        // a thread owns 4 CONSECUTIVE rows (pw*16 + r4*4 + i): when the chain boundaries are multiples of 4 (n = 168, 20, ...)
        // its rows all lie on one chain and it takes the selection-free path even in blocks that mix chains
        const int r4 = lane >> 3, c4 = lane & 7;
        const float4* const A4 = reinterpret_cast<const float4*>(g.A);
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        const int rofs = (int)rank * HROWS;        // this CTA's first row inside the 256-row block
        int ltile = pair, lkt = 0;
        bool lhave = ltile < num_tiles;
        uint32_t aoff[4];
        uint32_t lkinds = 0;                       // 2 bits per row: 0 upper, 1 lower, 2 Jacobian chain, 3 padding
        auto setup_load = [&]() {
            const PairGeo t = pair_geo(g, ltile, col_pairs, (int)rank);
            lkinds = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int j = rofs + pw * 16 + r4 * 4 + i;
                const int rin = t.rbase + j;
                int kind = rin / g.rows_kind;
                int rk = rin - kind * g.rows_kind;
                if (kind >= g.nkinds) { kind = 3; rk = 0; }
                aoff[i] = (uint32_t)(((size_t)(g.a_shared ? rk : (t.r0 + j)) * g.lda) >> 2) + c4;
                lkinds |= (uint32_t)kind << (2 * i);
            }
        };
        auto issue = [&](float4* buf, uint32_t& bkinds) {
            bkinds = lkinds;
            if (!lhave) return;
            const uint32_t ko = (uint32_t)lkt * (TBK / 4);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const bool ok = ((lkinds >> (2 * i)) & 3u) != 3u;
                buf[i] = ok ? __ldg(A4 + aoff[i] + ko) : zero4;
            }
            if (++lkt == nk) {
                lkt = 0;
                ltile += npairs;
                lhave = ltile < num_tiles;
                if (lhave) setup_load();
            }
        };
        int ptile = pair, pkt = 0;
        bool phave = ptile < num_tiles;
        PairGeo t_cur = pair_geo(g, phave ? ptile : 0, col_pairs, (int)rank);
        int stage = 0; uint32_t phase = 0;
        int ps = 0; uint32_t pphase = 0;
        auto lds4 = [&](uint32_t addr) {
            float4 v;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
            return v;
        };
        auto split_store = [&](const float4& v, uint32_t r_hi, uint32_t r_lo, int row) {
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
        float gsum[4] = {0.f, 0.f, 0.f, 0.f};
        auto step = [&](float4* P, uint32_t kP, float4* L, uint32_t& kL) -> bool {
            issue(L, kL);
            int ntile = ptile, nkt = pkt + 1;
            PairGeo t_nxt = t_cur;
            if (nkt == nk) { nkt = 0; ntile = ptile + npairs; }
            const bool nhave = ntile < num_tiles;
            if (nhave && nkt == 0) t_nxt = pair_geo(g, ntile, col_pairs, (int)rank);
            const bool do_gap = t_cur.rowsums && (g.gap != nullptr);
            float4 kUc, kLc, dpc = zero4, gU4 = zero4, gL4 = zero4;
            mbar_wait(bar_pfull(ps), pphase);
            const uint32_t pp = sP(ps) + c4 * 16;
            kUc = lds4(pp); kLc = lds4(pp + TBK * 4);
            if (g.nkinds == 3) dpc = lds4(pp + 2 * TBK * 4);
            if (do_gap) { gU4 = lds4(pp + 3 * TBK * 4); gL4 = lds4(pp + 4 * TBK * 4); }
            const int p_used = ps;
            if (++ps == PSTAGES) { ps = 0; pphase ^= 1; }
            mbar_wait(bar_rempty(stage), phase ^ 1);
            const uint32_t r_hi = sR(stage, 0), r_lo = sR(stage, 1);
            if (kP == 0u || kP == 0x55u || kP == 0xAAu || kP == 0xFFu) {
                // all four rows of this thread on one chain (upper / lower / Jacobian; padding rows are zero anyway)
                const bool jac = kP >= 0xAAu;
                const float4 kp = kP == 0u ? kUc : (jac ? dpc : kLc), kn = kP == 0u ? kLc : (jac ? dpc : kUc);
                const float4 gp = kP == 0u ? gU4 : (jac ? zero4 : gL4), gn = kP == 0u ? gL4 : (jac ? zero4 : gU4);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    float4 v = P[i];
                    if (do_gap) gsum[i] += gap4(v, gp, gn);
                    relax4(v, kp, kn);
                    split_store(v, r_hi, r_lo, pw * 16 + r4 * 4 + i);
                }
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    float4 v = P[i];
                    const uint32_t kind = (kP >> (2 * i)) & 3u;
                    if (kind < 2u) {
                        if (do_gap) gsum[i] += gap4(v, kind == 0u ? gU4 : gL4, kind == 0u ? gL4 : gU4);
                        relax4(v, kind == 0u ? kUc : kLc, kind == 0u ? kLc : kUc);
                    } else if (kind == 2u) {
                        relax4(v, dpc, dpc);
                    }
                    split_store(v, r_hi, r_lo, pw * 16 + r4 * 4 + i);
                }
            }
            // generic-proxy stores -> visible to the tensor core of the LEADER's SM (async proxy), then the hand-over
            // (one arrival per warp: every lane fences its own stores, the warp synchronises, lane 0 releases at cluster scope --
            // 256 remote arrivals per slab over the SM-to-SM network made the pair kernel slower than the single-CTA one)
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
                if (leader) mbar_arrive(bar_rfull(stage)); else mbar_arrive_remote(bar_rfull(stage), 0);
                mbar_arrive(bar_pempty(p_used));
            }
            if (++stage == R2STAGES) { stage = 0; phase ^= 1; }
            if (pkt == nk - 1) {
                if (do_gap) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        float s = gsum[i];
                        s += __shfl_xor_sync(0xffffffffu, s, 1);
                        s += __shfl_xor_sync(0xffffffffu, s, 2);
                        s += __shfl_xor_sync(0xffffffffu, s, 4);
                        const int m = t_cur.r0 + rofs + pw * 16 + r4 * 4 + i;
                        if (c4 == 0) g.gap[m] = (g.gap_init ? 0.f : g.gap[m]) + s;
                    }
                }
#pragma unroll
                for (int i = 0; i < 4; ++i) gsum[i] = 0.f;
            }
            ptile = ntile; pkt = nkt; t_cur = t_nxt;
            return nhave;
        };
        if (phave) {
            // four register buffers of 4 float4: the loads of a slab are issued three slabs before it is transformed
            float4 b0[4], b1[4], b2[4], b3[4];
            uint32_t k0 = 0, k1 = 0, k2 = 0, k3 = 0;
            setup_load();
            issue(b0, k0);
            issue(b1, k1);
            issue(b2, k2);
            while (true) {
                if (!step(b0, k0, b3, k3)) break;
                if (!step(b1, k1, b0, k0)) break;
                if (!step(b2, k2, b1, k1)) break;
                if (!step(b3, k3, b2, k2)) break;
            }
        }
    }

    // ---- teardown: the leader's MMAs read the peer's shared memory, so neither CTA may leave before both are done
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc_pair(tmem_base, TMEM_COLS);
    }
}

// ---------------------------------------------------------------------------------------------
// reverse-sweep step on CTA pairs: D_l = Lbar_{l-1} W_l^T with the sign-masked epilogue.  Same pair protocol
// as the forward; 768 threads per CTA: 4 control warps, 16 epilogue warps (bwd_epilogue_tile of nn_gemm_tc.cuh, this CTA's
// 128 output columns x all 256 rows, two alternating accumulators), 4 producer warps (this CTA's 128 rows, split only).
// ---------------------------------------------------------------------------------------------
constexpr int SMEM2B_BYTES = RING2_BYTES + 256;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS_BWD, 1)
chain_gemm_tc2_bwd_kernel(const GemmArgs g, const __grid_constant__ CUtensorMap tm_hi, const __grid_constant__ CUtensorMap tm_lo) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t sbase = smem_u32(smem_raw);
    if ((sbase & 1023u) != 0u) __trap();
    uint8_t* sgen = smem_raw;
    auto sW = [&](int s, int part) { return sbase + (2 * s + part) * W_TILE_BYTES; };
    auto sR = [&](int s, int part) { return sbase + WSTAGES * 2 * W_TILE_BYTES + (2 * s + part) * R2_TILE_BYTES; };
    const uint32_t bar0 = sbase + RING2_BYTES;
    auto bar_wfull = [&](int s) { return bar0 + 8 * s; };
    auto bar_wempty = [&](int s) { return bar0 + 8 * (WSTAGES + s); };
    auto bar_rfull = [&](int s) { return bar0 + 8 * (2 * WSTAGES + s); };
    auto bar_rempty = [&](int s) { return bar0 + 8 * (2 * WSTAGES + R2STAGES + s); };
    auto bar_tfull = [&](int a) { return bar0 + 8 * (2 * WSTAGES + 2 * R2STAGES + a); };
    auto bar_tempty = [&](int a) { return bar0 + 8 * (2 * WSTAGES + 2 * R2STAGES + 2 + a); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sgen + RING2_BYTES + 8 * (2 * WSTAGES + 2 * R2STAGES + 4));
    constexpr int kEpiWarps = 16, kProdWarps = 4, kEpiRows = TBN * 4 / kEpiWarps, RB = 8;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const bool leader = rank == 0;
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
    const int col_pairs = (g.N + 2 * TBM - 1) / (2 * TBM);
    const int row_blocks = g.M / TBN;
    const int num_tiles = row_blocks * col_pairs;
    const int nk = g.K / TBK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_hi);
        tma_prefetch_desc(&tm_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < WSTAGES; ++s) { mbar_init(bar_wfull(s), 1); mbar_init(bar_wempty(s), 1); }
        for (int s = 0; s < R2STAGES; ++s) { mbar_init(bar_rfull(s), 2 * kProdWarps); mbar_init(bar_rempty(s), 1); }
        for (int a = 0; a < 2; ++a) { mbar_init(bar_tfull(a), 1); mbar_init(bar_tempty(a), 2 * kEpiWarps); }
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc_pair(smem_u32(tmem_slot), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    // register pool of the CTA: 768 x 80 = 61 440 >= 128 x 40 (control) + 512 x 80 (epilogue) + 128 x 120 (producers)
    if (warp < 4) reg_dec<40>();
    if (warp == 0) {
        int stage = 0; uint32_t phase = 0;
        for (int tile = pair; tile < num_tiles; tile += npairs) {
            const PairGeo t = pair_geo(g, tile, col_pairs, (int)rank);
            for (int kt = 0; kt < nk; ++kt) {
                mbar_wait<32>(bar_wempty(stage), phase ^ 1);
                if (lane == 0) {
                    if (leader) mbar_arrive_expect_tx(bar_wfull(stage), 4 * W_TILE_BYTES);
                    tma_load_2d_pair(sW(stage, 0), &tm_hi, kt * TBK, t.n0, bar_wfull(stage));
                    tma_load_2d_pair(sW(stage, 1), &tm_lo, kt * TBK, t.n0, bar_wfull(stage));
                }
                __syncwarp();
                if (++stage == WSTAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        if (leader) {
            int ws = 0, rs = 0; uint32_t wphase = 0, rphase = 0;
            const uint32_t idesc = make_idesc(2 * TBM, TBN);
            const uint64_t dW0 = make_smem_desc(sW(0, 0)), dR0 = make_smem_desc(sR(0, 0));
            int tcount = 0;
            for (int tile = pair; tile < num_tiles; tile += npairs, ++tcount) {
                const int acc = tcount & 1;
                mbar_wait(bar_tempty(acc), ((tcount >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_main = tmem_base + acc * TBN;
                for (int kt = 0; kt < nk; ++kt) {
                    mbar_wait(bar_wfull(ws), wphase);
                    mbar_wait(bar_rfull(rs), rphase);
                    tc_fence_after();
                    const uint64_t whi = dW0 + (uint64_t)((2 * ws * W_TILE_BYTES) >> 4), wlo = whi + (W_TILE_BYTES >> 4);
                    const uint64_t rhi = dR0 + (uint64_t)((2 * rs * R2_TILE_BYTES) >> 4), rlo = rhi + (R2_TILE_BYTES >> 4);
                    if (lane == 0) {
#pragma unroll
                        for (int k = 0; k < TBK / 8; ++k) {
                            const uint64_t ko = (uint64_t)(k * 32 >> 4);
                            umma_tf32_pair(d_main, whi + ko, rlo + ko, idesc, (kt | k) != 0);
                            umma_tf32_pair(d_main, wlo + ko, rhi + ko, idesc, 1u);
                            umma_tf32_pair(d_main, whi + ko, rhi + ko, idesc, 1u);
                        }
                        umma_commit_pair(bar_wempty(ws));
                        umma_commit_pair(bar_rempty(rs));
                        if (kt == nk - 1) umma_commit_pair(bar_tfull(acc));
                    }
                    __syncwarp();
                    if (++ws == WSTAGES) { ws = 0; wphase ^= 1; }
                    if (++rs == R2STAGES) { rs = 0; rphase ^= 1; }
                }
            }
        }
    } else if (warp >= 4 && warp < 4 + kEpiWarps) {
        reg_dec<80>();                              // (keeps its 80 registers; without the statement ptxas spills 770 bytes here)
        const int q = warp & 3;
        const uint32_t t_lane = tmem_base + ((uint32_t)(q * 32) << 16);
        const int c_lo = ((warp - 4) >> 2) * kEpiRows, c_hi = c_lo + kEpiRows;
        int tcount = 0;
        for (int tile = pair; tile < num_tiles; tile += npairs, ++tcount) {
            const PairGeo t = pair_geo(g, tile, col_pairs, (int)rank);
            const int n = t.n0 + q * 32 + lane;
            const bool n_ok = n < g.N;
            const int acc = tcount & 1;
            const uint32_t tempty = bar_tempty(acc);
            bwd_epilogue_tile<RB, kEpiRows>(g, t.r0, t.rbase, t.po, n, n_ok, lane, t_lane + acc * TBN, c_lo, c_hi, bar_tfull(acc),
                                            (uint32_t)((tcount >> 1) & 1), [&]() {
                                                __syncwarp();
                                                if (lane == 0) { if (leader) mbar_arrive(tempty); else mbar_arrive_remote(tempty, 0); }
                                            });
        }
    } else if (warp >= 4 + kEpiWarps) {
        // ===================== row producers: this CTA's 128 rows, 8 rows per thread, split only =====================
        reg_inc<120>();
        const int pw = warp - (4 + kEpiWarps);
        const int r4 = lane >> 3, c4 = lane & 7;
        const float4* const A4 = reinterpret_cast<const float4*>(g.A);
        const uint32_t rstride = (uint32_t)(g.lda >> 2) * 4u;
        const int rofs = (int)rank * HROWS;
        int ltile = pair, lkt = 0;
        bool lhave = ltile < num_tiles;
        uint32_t lbase = 0;
        auto set_base = [&]() { lbase = (uint32_t)(((size_t)(ltile / col_pairs * TBN + rofs + pw * 32 + r4) * g.lda) >> 2) + c4; };
        auto issue = [&](float4* buf) {
            if (!lhave) return;
            const float4* src = A4 + lbase + (uint32_t)lkt * (TBK / 4);
#pragma unroll
            for (int i = 0; i < 8; ++i) buf[i] = __ldg(src + (size_t)i * rstride);
            if (++lkt == nk) {
                lkt = 0;
                ltile += npairs;
                lhave = ltile < num_tiles;
                if (lhave) set_base();
            }
        };
        int stage = 0; uint32_t phase = 0;
        long long remaining = 0;
        for (int tile = pair; tile < num_tiles; tile += npairs) remaining += nk;
        auto put = [&](const float4* buf) {
            mbar_wait(bar_rempty(stage), phase ^ 1);
            const uint32_t r_hi = sR(stage, 0), r_lo = sR(stage, 1);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float4 v = buf[i];
                float4 hi, lo;
                hi.x = to_tf32(v.x); hi.y = to_tf32(v.y); hi.z = to_tf32(v.z); hi.w = to_tf32(v.w);
                lo.x = v.x - hi.x; lo.y = v.y - hi.y; lo.z = v.z - hi.z; lo.w = v.w - hi.w;
                const int row = pw * 32 + i * 4 + r4;
                const uint32_t off = (uint32_t)row * 128u + (uint32_t)((c4 ^ (row & 7)) << 4);
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(r_hi + off), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w) : "memory");
                asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(r_lo + off), "f"(lo.x), "f"(lo.y), "f"(lo.z), "f"(lo.w) : "memory");
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) { if (leader) mbar_arrive(bar_rfull(stage)); else mbar_arrive_remote(bar_rfull(stage), 0); }
            if (++stage == R2STAGES) { stage = 0; phase ^= 1; }
        };
        if (lhave) {
            float4 b0[8], b1[8];
            set_base();
            issue(b0);
            while (true) {
                issue(b1); put(b0); if (--remaining == 0) break;
                issue(b0); put(b1); if (--remaining == 0) break;
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc_pair(tmem_base, TMEM_COLS);
    }
}

inline cudaError_t launch_chain_gemm_tc2_bwd(const GemmArgs& g, const CUtensorMap& hi, const CUtensorMap& lo, int num_sms, cudaStream_t st) {
    // the attribute is per device: one bit per device ordinal (a context may live on any GPU of the process)
    static std::atomic<unsigned long long> attr_done{0ull};
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned long long bit = 1ull << (dev & 63);
    if (!(attr_done.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(chain_gemm_tc2_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM2B_BYTES);
        if (e != cudaSuccess) return e;
        attr_done.fetch_or(bit, std::memory_order_release);
    }
    if (g.M % TBN != 0 || g.K % TBK != 0) return cudaErrorInvalidValue;
    const int tiles = (g.M / TBN) * ((g.N + 2 * TBM - 1) / (2 * TBM));
    int grid = 2 * tiles < num_sms ? 2 * tiles : (num_sms & ~1);
    chain_gemm_tc2_bwd_kernel<<<grid, THREADS_BWD, SMEM2B_BYTES, st>>>(g, hi, lo);
    return cudaGetLastError();
}

// g.M (coefficient rows) must be a multiple of 256, g.K a multiple of 32
inline cudaError_t launch_chain_gemm_tc2_fwd(const GemmArgs& g, const CUtensorMap& hi, const CUtensorMap& lo, int num_sms, cudaStream_t st) {
    // the attribute is per device: one bit per device ordinal (a context may live on any GPU of the process)
    static std::atomic<unsigned long long> attr_done{0ull};
    int dev = 0;
    cudaGetDevice(&dev);
    const unsigned long long bit = 1ull << (dev & 63);
    if (!(attr_done.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(chain_gemm_tc2_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM2_BYTES);
        if (e != cudaSuccess) return e;
        attr_done.fetch_or(bit, std::memory_order_release);
    }
    if (g.M % TBN != 0 || g.K % TBK != 0) return cudaErrorInvalidValue;
    const int tiles = (g.M / TBN) * ((g.N + 2 * TBM - 1) / (2 * TBM));
    int grid = 2 * tiles < num_sms ? 2 * tiles : (num_sms & ~1);
    chain_gemm_tc2_fwd_kernel<<<grid, THREADS, SMEM2_BYTES, st>>>(g, hi, lo);
    return cudaGetLastError();
}

}  // namespace tc2
}  // namespace leb_nn

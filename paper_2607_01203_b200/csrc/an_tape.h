// an_tape.h -- the interval tape of the analytic path (leb_analytic_fwd / leb_vjp kind 0).
//
// The path-based interval-Hessian bound (Thm 1, eq. (15)) needs, for every pair
// j <= k of coordinates of a = [x; u], the enclosure [H_{l,kj}](A^(j)) of all outputs l over the prefix
// box A^(j) (eq. (14)).  Reading R1 fixes the inclusion function: the natural
// interval extension of second-order forward-mode AD of the model's straight-line program, every
// SLP variable carrying the intervals (w, w_j, w_k, w_jk).
//
// Almost all of those jet components are STRUCTURALLY zero (config 4: 3.3e8 interval products per tile
// if evaluated densely, 2e6 that are not identically zero), and 0 * x = 0, 0 + x = x, 1 * x = x hold
// exactly under directed rounding.  So the model SLP is not evaluated by device code written per model:
// at leb_set_analytic time the host evaluates it SYMBOLICALLY (an_compile.cu: every jet component is
// `zero`, a constant, or a slot), emits only the interval operations that can be non-zero, removes what
// no output reads, and hands the device a tape.  The tape of one path index j is
//     segment WJ(j)  : the w and w_j components on A^(j)           (shared by every k >= j)
//     segments K(j,k): the w_k, w_jk components and the terms [H_kj] D_j D_k of eq. (15)
// in static single assignment form: instruction i of a segment writes slot (segment base + i).
// The device (analytic.cu) is an interpreter of that tape, one (trajectory, timestep) tile per lane,
// one (tile group, j) task per warp -- the tape is the same for every tile, so a warp never diverges --
// and its reverse sweep (adjoint slots, branch selections re-derived from the stored primal values) is
// the VJP.  No numerical step of the method runs on the host: the compiler handles structure only.
#pragma once
#include <stdint.h>
#include <vector>

namespace leb_an {

enum Op : uint32_t {
    OP_NOP = 0,
    OP_BOX,      // d = [nom[a] - rad[a], nom[a] + rad[a]]   (25a) L272, mu = 0;   b = gradient row of the task
    OP_PT,       // d = [nom[a], nom[a]]                      coordinates > j are pinned, L162
    OP_DELTA,    // d = [-rad[a], rad[a]]                     D = A (-) a~, L164
    OP_BOXMU,    // d = hull([nom + mu - rad, nom + mu + rad], nom)   non-centred box (25a), prefix hull (reading R4)
    OP_DELTAMU,  // d = [mu[a] - rad[a], mu[a] + rad[a]]
    OP_CONST,    // d = [c, c]                                b = float bits
    OP_ADD,      // d = a + b
    OP_SUB,      // d = a - b
    OP_NEG,      // d = -a
    OP_SCALE,    // d = c * a                                 b = float bits
    OP_ADDC,     // d = a + c                                 b = float bits
    OP_MUL,      // d = a * b       hull of the four endpoint products
    OP_SQR,      // d = a^2 >= 0
    OP_CUBE,     // d = a^3
    OP_RECIP,    // d = 1 / a       domain error if 0 in a
    OP_SIN,      // range-exact
    OP_COS,
    OP_OUT,      // acc[b & 0xffff] += a     (RD / RU);  b >> 16 = output index l (the VJP's cotangent)
    OP_MULACC,   // d = p + a * b   p = the result of the instruction just before (slot d - 1): the product and the sum are the
    OP_SCALEACC, // d = p + c * a   same two interval operations, fused by the compiler when the product has no other use
    OP_COUNT
};

// Instruction word: w0 = op (5 bits) | source of operand a (2 bits) | FAR (1 bit) | a (24 bits);
// w1 = operand b: slot (30 bits) | source of b (2 bits) for ADD / SUB / MUL, else float bits or a row.
// The interpreter keeps the last kRing results of a segment in shared memory (a ring indexed by slot % kRing) and the
// last one in registers.  Where an operand is read from is decided here, by the compiler: SRC_PREV (defined by the
// preceding instruction), SRC_RING (fewer than kRing instructions earlier in the same segment) or SRC_GLOBAL (the
// global slot file).  A slot whose value -- in the reverse sweep: whose adjoint -- is needed through the global file
// carries the FAR bit.
struct Ins { uint32_t w0, w1; };
constexpr uint32_t kRing = 64;
constexpr uint32_t OP_MASK = 31u, OP_FAR = 0x80u, SRC_SHIFT = 5, SRC_GLOBAL = 0, SRC_RING = 1, SRC_PREV = 2;
constexpr uint32_t B_MASK = 0x3fffffffu, B_SRC_SHIFT = 30;

inline uint32_t ins_op(const Ins& i) { return i.w0 & OP_MASK; }
inline uint32_t ins_a(const Ins& i) { return i.w0 >> 8; }

struct Seg { uint32_t begin, count; };          // instruction range in Tape::ins

struct Task {                                    // one path index j
    uint32_t j;
    uint32_t wj_begin, wj_count;                 // segment WJ(j); its slots are [0, wj_count)
    uint32_t seg_begin, seg_count;               // K segments (Tape::segs); their slots start at wj_count
    uint32_t n_slots;                            // wj_count + longest K segment
    uint32_t acc_base, n_acc;                    // rows of the partial-bound buffer (one per output this j touches)
    uint32_t grad_base, n_grad;                  // rows of the partial-gradient buffer (one per input this j reads)
    uint32_t cost;                               // instructions executed (forward)
};

// real FP32 operations per interval instruction (the algorithmic work the roofline counts; directed-rounding
// add / mul / fma and min / max count one each, sin / cos / rcp one each)
inline int op_flops(uint32_t op) {
    switch (op) {
        case OP_BOX: case OP_ADD: case OP_SUB: case OP_SCALE: case OP_ADDC: case OP_OUT: case OP_DELTAMU: return 2;
        case OP_BOXMU: return 4;
        case OP_MUL: return 14;
        case OP_MULACC: return 16;
        case OP_SCALEACC: return 4;
        case OP_SQR: return 5;
        case OP_CUBE: return 4;
        case OP_RECIP: return 2;
        case OP_SIN: case OP_COS: return 10;
        default: return 0;
    }
}

// A set of tasks with the fixed-order reduction tables that go with it.
struct TaskSet {
    std::vector<Task> tasks;                     // sorted by descending cost
    // bound l = sum of partial rows out_rows[out_ptr[l] .. out_ptr[l+1]) (ascending j)
    std::vector<uint32_t> out_ptr, out_rows;
    // gradient of input v = sum of partial-gradient rows var_rows[var_ptr[v] .. var_ptr[v+1])
    std::vector<uint32_t> var_ptr, var_rows;
    uint32_t acc_rows = 0, grad_rows = 0;
    uint64_t ins_fwd = 0;                        // instructions executed per tile, forward
};

struct Tape {
    int n = 0, N = 0;
    std::vector<Ins> ins;
    std::vector<Seg> segs;
    std::vector<Task> base;                      // one task per path index j, ascending j, rows not yet assigned
    std::vector<std::vector<uint32_t>> task_out, task_var;   // per base task: output index of each acc row, input of each grad row
    uint32_t max_slots = 0, max_acc = 0, max_grad = 0;
    uint64_t ins_fwd = 0;                        // instructions per tile, forward, one task per j
    double flops_fwd = 0.0;                      // algorithmic FP32 operations per tile, forward
    bool uses_mu = false;
};

// Task set for a launch: the base tasks, those longer than `target` instructions cut into several tasks -- the K segments
// of a task depend on WJ(j) only, so they can be dealt to several tasks that each re-run WJ(j).  The run time of a small
// batch is the longest task's; cutting trades a little repeated work for a shorter critical path.
void leb_build_taskset(const Tape& T, uint32_t target, TaskSet* set);

}  // namespace leb_an

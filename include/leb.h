/* leb.h -- C ABI of the B200-native linearization-error-bound (LEB) library.
 *
 * What the library computes (arxiv/paper_2607_01203, "GPUSLS-LEO"; citations are
 * PAPER.md line numbers): for every trajectory b, timestep t (a "tile") and state
 * dimension i, a sound enclosure [r_lo, r_hi] of the linearization remainder
 *
 *     r_i(a) = f_i(a) - f_i(a~) - J(a~)(a - a~),   a = [x; u] in the tube box A_t     (10) L133
 *
 * where A_t = a~ + mu + [-sigma, sigma] is the tube box (25a) L272 (mu = NULL: the centred box, mu = 0),
 *   - for analytic dynamics by the path-based interval-Hessian bound, Thm 1 eq. (15);
 *   - for MLP dynamics by CROWN affine relaxations (Thm 2, eq. (18)) followed by the
 *     local Jacobian correction and box concretisation of Thm 3, eq. (19)-(21) L204-220;
 * the vector-Jacobian product of those bounds with respect to the nominal point a~ and the
 * radii sigma (differentiability, Sec. IV-D; consumed by J_err (35) L358-362); and the
 * fold of the per-dimension bounds into the non-zero-centred disturbance zonotope
 * (c_bar, R_bar), Sec. IV-C, eq. (25b,c) L274-281, diagonal padding L347.
 *
 * Conventions (all entry points):
 *   - extern "C", no exceptions cross the boundary, every call returns a leb_status.
 *   - Data pointers are DEVICE pointers owned by the caller unless the call is given
 *     LEB_FLAG_HOST_IO, in which case they are HOST pointers (pinned memory recommended) and the
 *     library stages them through its own device buffers (H2D before, D2H after, same stream).
 *     The library never frees caller memory and keeps no caller pointer after the call returns
 *     (leb_set_mlp copies and re-packs the weights into memory the context owns).
 *   - Calls are asynchronous on the caller's stream (`stream` is a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  Argument / shape errors are reported
 *     synchronously; CUDA launch errors surface as LEB_ERR_CUDA.
 *   - All arrays are FP32, row-major.  Trajectory arrays are [B, T, ld] with the row stride
 *     `ld_in` (>= N = n + m) or `ld_out` (>= n) given in floats; tile (b, t) is row b*T + t.
 *     Augmented-state order is a = [x; u] (state first, L131); this fixes the path order of (15).
 *   - A tile whose inputs are outside the method's domain (NaN/Inf input, sigma < 0, or an
 *     analytic box on which cos(theta) contains 0, so 1/cos is unbounded) gets r_lo = -inf,
 *     r_hi = +inf for all its dimensions and raises the context's domain flag, readable after
 *     synchronising the stream with leb_domain_flag().  A finite bound is never silently wrong.
 *   - An empty batch (B == 0 or T == 0) is legal: the call returns LEB_OK, launches nothing and
 *     does not look at the data pointers (they may be NULL).
 *   - There is no CPU fallback: every numerical step runs in the library's sm_100a kernels.
 */
#ifndef LEB_H_
#define LEB_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct leb_ctx leb_ctx; /* opaque: packed weights, workspace, staging buffers, flags */

typedef enum {
    LEB_OK = 0,
    LEB_ERR_ARG = 1,         /* NULL pointer, negative size, unknown enum value */
    LEB_ERR_SHAPE = 2,       /* ld too small, model/shape mismatch */
    LEB_ERR_ALIGN = 3,       /* pointer not 4-byte aligned */
    LEB_ERR_DOMAIN = 4,      /* reported by leb_domain_flag(): some tile hit a domain error */
    LEB_ERR_UNSUPPORTED = 5, /* unknown model; certified mode with layers wider than 2048 */
    LEB_ERR_CUDA = 6,
    LEB_ERR_NOMEM = 7,
    LEB_ERR_STATE = 8,       /* model not set before the call that needs it */
    LEB_ERR_CAPACITY = 9     /* problem larger than a fixed-capacity entry point holds (leb_jerr_static: B * T > LEB_JERR_STATIC_MAX) */
} leb_status;

typedef enum { LEB_MODEL_UNICYCLE = 1, LEB_MODEL_QUAD12 = 2, LEB_MODEL_QUADCHAIN = 3, LEB_MODEL_PLANAR_QUAD = 4,
               LEB_MODEL_SATELLITE = 5, LEB_MODEL_QUADCENTROID = 6 } leb_model_id;
typedef enum { LEB_INTEG_EULER = 1, LEB_INTEG_RK4 = 2 } leb_integ;
typedef enum { LEB_ACT_RELU = 1, LEB_ACT_TANH = 2 } leb_act;

/* Analytic dynamics.
 *   UNICYCLE : a = (px, py, th, v, om); f = (px + dt v cos th, py + dt v sin th, th + dt om).
 *   QUAD12   : xi = (p[3], (phi, theta, psi), v[3], (p, q, r)) -- state order of L538 --,
 *              nu = (T, tau[3]); ZYX rigid-body vector field (eq. (38), de-garbled).
 *   QUADCHAIN: n_units copies of QUAD12, x = (xi_1..xi_U), u = (nu_1..nu_U) ((39) L540-543),
 *              neighbours joined per axis by the spring k1 d + k3 d^3 (BASELINE config 4).
 *   PLANAR_QUAD: x = (px, py, phi, vx, vy, phidot), u = (u1, u2), eq. (37a);
 *              mass = m, g, Jx = moment of inertia J, k1 = arm length L.
 *   SATELLITE: x = (q[4], om[3]), u = torque[3], eq. (36); (Jx, Jy, Jz) = diag of I_S.
 *   QUADCENTROID: n_units copies of QUAD12 with the paper's centroid spring-damper coupling (40)-(42) L545-558;
 *              k1 = alpha (stiffness), k3 = gamma (damping).
 * integ = EULER: f = x + dt g(x,u) (the paper's choice, L505); RK4: classical 4 stages, u held. */
typedef struct {
    int model_id; /* leb_model_id */
    int integ;    /* leb_integ (UNICYCLE is always Euler) */
    int n_units;  /* QUADCHAIN: number of quadrotors (config 4: 14); otherwise 1 */
    float dt, mass, g, Jx, Jy, Jz, k1, k3;
} leb_analytic_model;

/* MLP dynamics f(x,u) = x + g(x,u) if residual else g(x,u);
 * g(a) = W_L phi(... phi(W_1 a + b_1) ...) + b_L.  The residual term is linear, so the
 * remainder of f equals the remainder of g (reading R10). */
typedef struct {
    int n_layers;          /* L = number of weight matrices (hidden layers = L-1 >= 1) */
    const int* dims;       /* HOST array of L+1 ints: dims[0] = n+m ... dims[L] = n */
    const float* const* W; /* HOST array of L pointers; W[l] is [dims[l+1], dims[l]] row-major */
    const float* const* b; /* HOST array of L pointers; b[l] is [dims[l+1]] */
    int act;               /* leb_act */
    int residual;          /* 0/1 (informational: does not change the bounds) */
    int weights_on_host;   /* 0: W[l], b[l] point to device memory; 1: host memory */
} leb_mlp;

enum {
    LEB_FLAG_NO_MARGIN = 1u, /* NN: value mode -- plain FP32 / 3xTF32 result with no rounding margin (the mode the
                                parity tests compare with the oracle).  Without it leb_nn_fwd runs in CERTIFIED mode:
                                every rounding error of the path is bounded and added outward,
                                so r_lo <= r(a) <= r_hi holds in exact arithmetic for the FP32 weights as given */
    LEB_FLAG_FFMA_ONLY = 2u, /* NN: FP32 FFMA contractions instead of 3xTF32 tcgen05 */
    LEB_FLAG_HOST_IO = 4u,   /* data pointers of this call are host pointers */
    LEB_FLAG_SINGLE_CTA = 16u, /* NN: forward chain steps on single CTAs (nn_gemm_tc.cuh) instead of CTA pairs
                                  (tcgen05.mma.cta_group::2, nn_gemm_tc2.cuh, the default); same results bit for bit */
    LEB_FLAG_IBP_HIDDEN = 32u, /* NN: CROWN-IBP -- the bounds of hidden layers 2..L-1 by interval propagation of the previous
                                  layer's bounds instead of back-substitution (about 4x fewer flops at config 5, looser
                                  bounds); the output is back-substituted as always.  Certified mode: the interval
                                  propagation is the non-centred layer-1 formula applied to the activation deviations,
                                  every |W| product rounded up.  leb_vjp takes the same flag. */
    LEB_FLAG_REUSE_FWD = 8u  /* leb_vjp(kind 1) becomes STATEFUL: the caller states that (nom, rad) are those of the previous
                                leb_nn_fwd call on this context (J == NULL).  If the workspace still holds that call's complete
                                forward state (the batch fitted one chunk) AND that state was computed in the mode this
                                leb_vjp call names (LEB_FLAG_NO_MARGIN set: a value-mode forward; clear: a certified one), the
                                reverse sweep starts from it instead of recomputing the forward.  Otherwise the flag has no
                                effect: the call recomputes a value-mode forward, exactly as the stateless call does.
                                leb_nn_state() reports which of the two happened.  Reverse sweep over a CERTIFIED state: the
                                derivative of the value-mode formulas evaluated on the certified forward's (widened) hidden
                                bounds and padded gaps, i.e. the gradient of the certified bound with its rounding pads and
                                outward-rounding factors (<= 3e-4 relative) treated as constants. */
};

leb_status leb_create(leb_ctx** ctx, int device);
leb_status leb_destroy(leb_ctx* ctx);
const char* leb_status_str(leb_status s);

/* Select the analytic model used by leb_analytic_fwd / leb_vjp(kind 0). */
leb_status leb_set_analytic(leb_ctx* ctx, const leb_analytic_model* model);

/* Copy, pad and pre-split the MLP weights into context-owned device memory (done once per
 * model; enqueued on `stream`).  Used by leb_nn_fwd / leb_vjp(kind 1). */
leb_status leb_set_mlp(leb_ctx* ctx, const leb_mlp* mlp, void* stream);

/* Upper bound, in tiles, of the batch slice processed at once by the NN path (bounds the
 * workspace: the forward keeps every back-substituted coefficient block of the slice in HBM).
 * 0 restores the default.  Does not change results. */
leb_status leb_set_nn_chunk(leb_ctx* ctx, int tiles_per_chunk);

/* Path-based interval-Hessian bound, Thm 1 eq. (15), for every tile.
 *   nom, rad : [B, T, ld_in]  nominal a~ and radii sigma >= 0
 *   mu       : NULL (centred box) or [B, T, ld_in]: the box is a~ + mu + [-sigma, sigma] (25a) L272, D = A (-) a~ =
 *              [mu - sigma, mu + sigma] (L164), and the Hessian enclosures of (15) are taken on the prefix sets of
 *              hull(A u {a~}) (reading R4: Thm 1 needs the whole segment from a~ to a point of A)
 *   r_lo,r_hi: [B, T, ld_out] outputs, r_lo <= r(a) <= r_hi on the box, outward-rounded FP32. */
leb_status leb_analytic_fwd(leb_ctx* ctx, int B, int T, const float* nom, const float* rad,
                            const float* mu, int ld_in, float* r_lo, float* r_hi, int ld_out,
                            unsigned flags, void* stream);

/* Input-domain partitioning (Sec. IV-D): the box of every tile is cut into a grid of sub-boxes, splits[g] >= 1 equal
 * parts along coordinate g (HOST array of N ints; at most 65536 sub-boxes per tile); every sub-box is bounded as a
 * non-centred box about the same nominal point and the hull of the sub-box enclosures is returned.  Sound (every point of
 * the box lies in a sub-box; FP32 sub-boxes are padded to overlap) and never wider than leb_analytic_fwd's enclosure
 * (inclusion isotonicity).  Other arguments as leb_analytic_fwd. */
leb_status leb_analytic_partition_fwd(leb_ctx* ctx, int B, int T, const float* nom, const float* rad, const float* mu,
                                      int ld_in, const int* splits, float* r_lo, float* r_hi, int ld_out,
                                      unsigned flags, void* stream);

/* VJP of leb_analytic_partition_fwd: the hull takes each bound from one sub-box (the first minimum / maximum in sub-box
 * order, reading R20), so the cotangent of an output goes to that sub-box's bound, through the ordinary reverse sweep, and
 * back through the sub-box construction (radius sigma / splits, offset mu + sigma c_p) to nom, rad and mu.  Recomputes the
 * sub-box forward (stateless).  g_lo, g_hi: [B, T, ld_out]; grad_nom, grad_rad (, grad_mu when mu != NULL): [B, T, ld_in]. */
leb_status leb_analytic_partition_vjp(leb_ctx* ctx, int B, int T, const float* nom, const float* rad, const float* mu,
                                      int ld_in, const int* splits, const float* g_lo, const float* g_hi, int ld_out,
                                      float* grad_nom, float* grad_rad, float* grad_mu, unsigned flags, void* stream);

/* Nominal-point refinement by projected gradient descent (Sec. IV-D, Table II).  The box of every tile is
 * FIXED (centre, rad); the nominal point a~ moves inside |a~ - centre| <= eps (componentwise) so as to shrink the total
 * width W(a~) = sum_i (r_hi_i - r_lo_i) of the enclosure of the remainder about a~ on that box (mu = centre - a~).
 * `steps` plain gradient steps a~ <- proj(a~ - lr dW/da~) (the paper gives no step rule: DESIGN.md reading R22), all on
 * the device; the best iterate is kept.
 *   centre, rad, eps : [B, T, ld_in]
 *   nom              : [B, T, ld_in] in: starting points (inside the neighbourhood); out: best nominal points
 *   width0, width    : [B, T] total width at the start / at the returned point */
leb_status leb_analytic_pgd(leb_ctx* ctx, int B, int T, const float* centre, const float* rad, const float* eps, int ld_in,
                            int steps, float lr, float* nom, float* width0, float* width, unsigned flags, void* stream);

/* CROWN + Thm 3 bound, eq. (18)-(21) L196-220, for every tile.
 *   mu     : NULL (centred box) or [B, T, ld_in]: the box is a~ + mu + [-sigma, sigma] (25a) L272; the CROWN bounds are
 *            taken on that box, p(a~) and J(a~) stay at the nominal point, and (21) maximises the affine bound (20) over
 *            the box (in the kernels' deviation form: a - a~ in mu -+ sigma).  Certified mode keeps its guarantee: the
 *            layer-1 shift W_1 mu and the Lam_0 mu sums are padded outward like every other sum; the relaxation
 *            gaps stay at zhat(a~), clamped to gU >= 0 >= gL, which is sound and up to a few % wider than value
 *            mode when |W_1 mu| exceeds a neuron's radius.
 *   J      : NULL => the network's own Jacobian at a~ (eq. (7)); otherwise [B, T, n, N]
 *            dense, and the bound is with respect to that matrix (Thm 3 holds for any J).
 *   margin : NULL or [B, T, ld_out].  Certified mode: the outward pad contained in r_lo / r_hi of the entry (the
 *            larger of the two sides): rounding pads of the output rows' chain steps, the nominal drift eta and the
 *            rounding of the final sums.  (The pads of the hidden-layer bounds act through looser relaxations and
 *            are not part of this number; certified minus value-mode bound is the total cost.)  Value mode: 0.
 * Certified mode returns LEB_ERR_UNSUPPORTED for layers wider than 2048 (padded). */
leb_status leb_nn_fwd(leb_ctx* ctx, int B, int T, const float* nom, const float* rad,
                      const float* mu, const float* J, int ld_in, float* r_lo, float* r_hi,
                      float* margin, int ld_out, unsigned flags, void* stream);

/* CROWN with optimisable lower slopes (alpha-CROWN style; the paper names CROWN only, L194-196).  ReLU
 * networks: the lower line of an unstable neuron (l < 0 < u) is alpha z with ANY alpha in [0, 1].  Starting from the adaptive
 * choice of leb_nn_fwd, `steps` projected gradient steps alpha <- clip(alpha - lr dW/dalpha, 0, 1) on the total width
 * W = sum_i (r_hi_i - r_lo_i) of each tile's enclosure (one slope set per tile; dW/dalpha comes from the ordinary reverse
 * sweep), all on the device; every iterate is a sound enclosure and the tightest one per tile is returned.
 * The descent runs on the plain FP32 bound; the kept slopes are then evaluated once more in the mode `flags` names --
 * certified by default (the certificate of leb_nn_fwd holds for any lower slope in [0, 1]) -- and that is what is returned.
 * The forward state of this last evaluation stays resident: leb_vjp(kind 1, LEB_FLAG_REUSE_FWD, same mode flags) then
 * returns the gradient of the REFINED bound with the kept slopes held constant (a stateless leb_vjp differentiates the
 * adaptive-slope bound of leb_nn_fwd).  tanh networks, LEB_FLAG_IBP_HIDDEN: LEB_ERR_UNSUPPORTED.
 *   width0, width : [B, T] total width of the adaptive-slope enclosure (plain FP32 bound, what the descent starts from) /
 *                   of the returned one (in the mode `flags` names).  Other arguments as leb_nn_fwd. */
leb_status leb_nn_alpha_fwd(leb_ctx* ctx, int B, int T, const float* nom, const float* rad, int ld_in, int steps, float lr,
                            float* r_lo, float* r_hi, int ld_out, float* width0, float* width, unsigned flags, void* stream);

/* VJP of the bounds: grad = d/d(a~, sigma) sum_i g_hi[i] r_hi[i] + g_lo[i] r_lo[i], per tile
 * (block-diagonal over tiles).  Stateless by default: the forward pass is recomputed internally, and for kind 1 it
 * is recomputed in value mode whatever the flags say -- the certified margin is a rounding-level pad and is treated
 * as a constant.  The one stateful variant is LEB_FLAG_REUSE_FWD (see the flag).
 * Reproducibility: both kinds reduce in a fixed order except the NN reverse sweep's column sums (FP32 atomicAdd, one
 * per column and row block), so kind-1 gradients repeat to ~1e-6 relative, kind-0 gradients bit for bit.
 *   kind: 0 analytic (model from leb_set_analytic), 1 NN (model from leb_set_mlp)
 *   g_lo, g_hi       : [B, T, ld_out] cotangents
 *   grad_nom,grad_rad: [B, T, ld_in] outputs (columns >= N are left untouched).
 * min / max / abs / ReLU-switch / relaxation-case selections are treated as branch selections
 * (derivative of the selected branch), as in DESIGN.md "VJP definition". */
leb_status leb_vjp(leb_ctx* ctx, int kind, int B, int T, const float* nom, const float* rad,
                   const float* g_lo, const float* g_hi, int ld_in, int ld_out, float* grad_nom,
                   float* grad_rad, unsigned flags, void* stream);

/* leb_vjp for non-centred boxes: the same, with the box offsets mu [B, T, ld_in] as a third argument of the bound and
 * its gradient grad_mu [B, T, ld_in] as a third output (grad_mu may be NULL).  mu == NULL: identical to leb_vjp.
 * Both kinds (kind 1: the gradient of the value-mode bound). */
leb_status leb_vjp_mu(leb_ctx* ctx, int kind, int B, int T, const float* nom, const float* rad, const float* mu,
                      const float* g_lo, const float* g_hi, int ld_in, int ld_out, float* grad_nom,
                      float* grad_rad, float* grad_mu, unsigned flags, void* stream);

/* Zonotope fold, L229-231 and (25b,c) L274-281: c_bar = (r_lo + r_hi)/2,
 * R_diag = (r_hi - r_lo)/2 + pad (padding L347), rounded so that
 * [r_lo, r_hi] is contained in [c_bar - R_diag, c_bar + R_diag] in FP32.
 *   r_lo, r_hi, c_bar, R_diag : [B, T, n] contiguous
 *   E_diag     : NULL or [n], the (constant, diagonal) disturbance matrix E
 *   Ebar_dense : NULL or [B, T, n, 2n]: E_bar = [diag(E)  diag(R_diag)]  (25b) */
leb_status leb_zonotope_inflate(leb_ctx* ctx, int B, int T, int n, const float* r_lo,
                                const float* r_hi, const float* E_diag, float pad, float* c_bar,
                                float* R_diag, float* Ebar_dense, unsigned flags, void* stream);

/* Cotangents of (c_bar, R_diag) -> cotangents of (r_lo, r_hi) (the fold is linear):
 * g_lo = (gc - gR)/2, g_hi = (gc + gR)/2.  Arrays [B, T, n] contiguous. */
leb_status leb_zonotope_inflate_vjp(leb_ctx* ctx, int B, int T, int n, const float* gc,
                                    const float* gR, float* g_lo, float* g_hi, unsigned flags,
                                    void* stream);

/* Disturbance-error enclosure, eq. (22): r_dist = (E(x) - E_k) w in ([E](Omega^x) (-) E_k) E_nw, added IN PLACE to
 * the linearization-error enclosure (r = r_lin + r_dist, L228), outward rounded.  The caller supplies the interval
 * enclosure of the disturbance matrix over the state tube (the paper's systems all have constant E, for which this
 * call adds nothing).
 *   E_lo, E_hi, E_nom : [B, T, n, nw]  E_lo <= E(x) <= E_hi on the tube, E_nom = E(z_k)
 *   r_lo, r_hi        : [B, T, n] contiguous, updated */
leb_status leb_dist_add(leb_ctx* ctx, int B, int T, int n, int nw, const float* E_lo, const float* E_hi,
                        const float* E_nom, float* r_lo, float* r_hi, unsigned flags, void* stream);

/* Tube propagation, eq. (27)-(28) L289-291: for k = 1..T
 *     h_mu_k = sum_{j<k} Phi_{k,j} c_bar_j,   h_sigma_k = sum_{j<k} || Phi_{k,j} [diag(E) diag(R_bar_j)] ||_{1,r}
 * (row-wise 1-norm; every operation of h_sigma rounded up: it is a bound).
 *   Phi          : [B, T (T+1) / 2, N, n], N = n + m: block (k-1) k / 2 + j holds Phi_{k,j} = [Phi^x; Phi^u], 0 <= j < k <= T
 *   c_bar, R_diag: [B, T, n] (leb_zonotope_inflate's outputs);  E_diag: [n] or NULL (= 0)
 *   h_mu, h_sigma: [B, T, N], row k-1 = time k.   n > 8192: LEB_ERR_UNSUPPORTED. */
leb_status leb_tube_propagate(leb_ctx* ctx, int B, int T, int n, int m, const float* Phi, const float* c_bar,
                              const float* R_diag, const float* E_diag, float* h_mu, float* h_sigma,
                              unsigned flags, void* stream);

/* Propagated-error penalty, eq. (35) L360 (the sum over k read as k = j+1..T: Phi_{j,j} does not exist in (26)-(28)):
 *     J_err[b] = sum_j sum_{k>j} || Phi_{k,j} [diag(E) diag(R_bar_j)] ||_F^2,   grad_R = d J_err / d R_diag [B, T, n]
 * grad_R (may be NULL) is the cotangent gR of leb_zonotope_inflate_vjp, which leb_vjp then takes to (a~, sigma).
 *   J_err : [B].   n > 1024: LEB_ERR_UNSUPPORTED. */
leb_status leb_jerr(leb_ctx* ctx, int B, int T, int n, int m, const float* Phi, const float* R_diag,
                    const float* E_diag, float* J_err, float* grad_R, unsigned flags, void* stream);

/* leb_jerr for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same operation, same kernels, same results, but the per-(b, j) partial sums go to a static device array
 * of LEB_JERR_STATIC_MAX floats (256 KB, held by every GPU that loads the library until the process exits) instead of a
 * buffer from cudaMalloc.  The call makes no cudaMalloc / cudaFree / allocating library call and records no event.
 *   - device pointers only: LEB_FLAG_HOST_IO => LEB_ERR_ARG (host staging would have to allocate);
 *   - B * T > LEB_JERR_STATIC_MAX => LEB_ERR_CAPACITY, nothing is launched;
 *   - the array is shared by every call on the device and keeps the last call's contents (nothing in it has to start at
 *     zero: each call writes every entry it reads); calls that overlap on the GPU -- two streams, two contexts on one
 *     device -- RACE on it: serialise them (one stream, or an event between them).
 * Other arguments and errors as leb_jerr. */
#define LEB_JERR_STATIC_MAX 65536
leb_status leb_jerr_static(leb_ctx* ctx, int B, int T, int n, int m, const float* Phi, const float* R_diag,
                           const float* E_diag, float* J_err, float* grad_R, unsigned flags, void* stream);

/* *flag = 1 if any tile of any call since the last leb_domain_flag() hit a domain error
 * (synchronises `stream`, then clears the flag). */
leb_status leb_domain_flag(leb_ctx* ctx, int* flag, void* stream);

/* Inspection (tests): pre-activation bounds (l_s, u_s) of hidden layer `layer` (1-based) left
 * in the workspace by the LAST leb_nn_fwd call whose B*T fitted one chunk.
 * l, u: device [B*T, dims[layer]] contiguous. */
leb_status leb_nn_hidden_bounds(leb_ctx* ctx, int layer, float* l, float* u, void* stream);

/* Inspection (tests): the back-substituted coefficient rows Lambda_0 (coefficients on the input a = [x; u],
 * eq. (18)) of target layer `target` (2 .. L; L = the output target) left in the workspace by the
 * LAST leb_nn_fwd call whose B*T fitted one chunk.  out: device [B*T, 2, rows, dims[0]] contiguous, rows =
 * dims[target]; index 0 = upper chain, 1 = lower chain.  Used to measure the contraction's rounding error
 * against the model behind the certified margin. */
leb_status leb_nn_chain_coeffs(leb_ctx* ctx, int target, float* out, void* stream);

/* Inspection: the relaxation slopes (k^U, k^L of (18) PAPER.md:L196-200) of hidden layer `layer` (1-based) in the forward
 * state the LAST leb_nn_fwd / leb_nn_alpha_fwd call left (B*T fitted one chunk).  After leb_nn_alpha_fwd the lower slopes of
 * the unstable neurons are the refined ones.  kU, kL: device [B*T, dims[layer]] contiguous. */
leb_status leb_nn_slopes(leb_ctx* ctx, int layer, float* kU, float* kL, void* stream);

/* The Jacobian J~ the LAST leb_nn_fwd call with J == NULL subtracted in (20) PAPER.md:L209 -- the network's Jacobian at a~
 * (eq. (7)) as the library's own chain computed it, rounding included.  The certified enclosure is an enclosure of
 * p(a) - p(a~) - J~ (a - a~) for exactly this matrix, so a caller that linearises with it inherits the guarantee.
 * out: device [B*T, n, N] contiguous.  LEB_ERR_STATE if no such forward is resident (B*T larger than one chunk, or the
 * last forward was given the caller's J). */
leb_status leb_nn_jacobian(leb_ctx* ctx, float* out, void* stream);

/* State of the NN workspace (host-side query, no synchronisation): *tiles = number of tiles whose complete forward
 * state the last leb_nn_fwd / leb_vjp left resident (0: none, e.g. the batch was processed in chunks); *certified =
 * 1 if that state is a certified-mode one; *vjp_reused = 1 if the last leb_vjp(kind 1) call started from the
 * resident state (LEB_FLAG_REUSE_FWD honoured), 0 if it recomputed the forward. */
leb_status leb_nn_state(leb_ctx* ctx, int* tiles, int* certified, int* vjp_reused);

/* Statistics of the analytic model's interval tape (host-side query; roofline bookkeeping):
 * *flops_per_tile = FP32 operations of one forward pass over one tile (directed-rounding add / mul, min / max, one
 * per sin / cos / reciprocal), *ins_per_tile = interval instructions executed per tile (forward), *tape_ins =
 * instructions stored, *tasks = path indices j with any non-zero Hessian entry, *max_slots = slots of the largest task. */
leb_status leb_analytic_tape_stats(leb_ctx* ctx, double* flops_per_tile, long long* ins_per_tile, long long* tape_ins,
                                   int* tasks, int* max_slots);

/* Number of kernel launches the library has enqueued on this context so far. */
long long leb_launch_count(const leb_ctx* ctx);

/* Measurement aid (bench.py "roofline"): while enabled, every launch of
 * the library's kernels is bracketed by CUDA events on the launching stream.  Kernel classes:
 * 0 CROWN chain contraction (forward), 1 chain contraction (reverse sweep), 2 analytic forward,
 * 3 analytic VJP, 4 zonotope fold, 5 other NN kernels' GEMMs, 6 disturbance error / tube propagation / J_err.
 * leb_profile_read synchronises `stream` and returns, for one class and since the last
 * leb_profile_reset: the summed device time in ms, the summed ALGORITHMIC work (classes 0, 1, 5: flops computed
 * from the true, unpadded shapes; class 2: the tape's FP32 operations; class 3: three times that, the reverse sweep
 * counted as twice the forward; classes 4, 6: bytes) and the launch count. */
leb_status leb_profile(leb_ctx* ctx, int enable);
leb_status leb_profile_read(leb_ctx* ctx, int kernel_class, double* ms, double* work, long long* launches,
                            void* stream);
leb_status leb_profile_reset(leb_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LEB_H_ */

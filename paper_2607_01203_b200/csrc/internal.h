// internal.h -- declarations shared by the translation units of libleb.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include "../../include/leb.h"

#include <vector>

namespace leb_an {
struct Tape;
// analytic model with its derived constants (leb_make_model)
struct Model {
    int id, integ, n_units, n, N;
    float dt, half_dt, dt6;                      // dt, dt/2, dt/6
    float inv_m, g, cp, cq, cr, iJx, iJy, iJz;   // 1/m, g, (Jy-Jz)/Jx, (Jz-Jx)/Jy, (Jx-Jy)/Jz, 1/J*
    float k1, k3;                                // chain spring; planar quadrotor: k1 = arm length / inertia
};
void leb_compile_tape(const Model& M, bool with_mu, Tape* T);      // an_compile.cu (host, structure only)
}

// ---- profiling aid (leb_profile / leb_profile_read): CUDA events around the launches of each
// kernel class, on the launching stream, so that bench.py can report the dominant kernel's average
// launch duration measured live over the timed region.
enum { LEB_KC_CHAIN_FWD = 0, LEB_KC_CHAIN_BWD = 1, LEB_KC_ANALYTIC_FWD = 2, LEB_KC_ANALYTIC_VJP = 3,
       LEB_KC_INFLATE = 4, LEB_KC_NN_OTHER = 5, LEB_KC_TUBE = 6, LEB_KC_COUNT = 7 };
struct LebProf {
    bool on = false;
    struct Rec { cudaEvent_t a, b; int kc; };
    std::vector<Rec> recs;        // pool (events are reused after leb_profile_read)
    size_t used = 0;
    double work[LEB_KC_COUNT] = {0};   // algorithmic flops (or bytes for LEB_KC_INFLATE)
    long long count[LEB_KC_COUNT] = {0};
    void begin(int kc, cudaStream_t st) {
        if (!on) return;
        if (used == recs.size()) {
            Rec r{};
            cudaEventCreate(&r.a);
            cudaEventCreate(&r.b);
            recs.push_back(r);
        }
        recs[used].kc = kc;
        cudaEventRecord(recs[used].a, st);
    }
    void end(int kc, cudaStream_t st, double w) {
        if (!on) return;
        cudaEventRecord(recs[used].b, st);
        ++used;
        work[kc] += w;
        ++count[kc];
    }
    void destroy() {
        for (auto& r : recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
        recs.clear();
        used = 0;
    }
};

// ---- analytic path (analytic.cu: interpreter of the interval tape compiled by an_compile.cu)
struct AnState;   // model, tapes (host + device), workspace; owned by the context
leb_an::Model leb_make_model(const leb_analytic_model& m);
AnState* leb_an_create();
void leb_an_destroy(AnState*);
bool leb_an_ready(const AnState*);
int leb_an_n(const AnState*);
int leb_an_N(const AnState*);
leb_status leb_an_set_model(AnState*, const leb_an::Model& M);
leb_status leb_an_forward(AnState*, int tiles, const float* nom, const float* rad, const float* mu, int ld_in, float* r_lo,
                          float* r_hi, int ld_out, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof);
leb_status leb_an_vjp(AnState*, int tiles, const float* nom, const float* rad, const float* mu, const float* g_lo,
                      const float* g_hi, int ld_in, int ld_out, float* grad_nom, float* grad_rad, float* grad_mu,
                      int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof);
leb_status leb_an_partition(AnState*, int tiles, const float* nom, const float* rad, const float* mu, int ld_in,
                            const int* splits_host, float* r_lo, float* r_hi, int ld_out, int* domain_flag, cudaStream_t st,
                            long long* launches, LebProf* prof);
leb_status leb_an_partition_vjp(AnState*, int tiles, const float* nom, const float* rad, const float* mu, int ld_in,
                                const int* splits_host, const float* g_lo, const float* g_hi, int ld_out, float* grad_nom,
                                float* grad_rad, float* grad_mu, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof);
leb_status leb_an_pgd(AnState*, int tiles, const float* centre, const float* rad, const float* eps, int ld_in, int steps, float lr,
                      float* nom, float* w0, float* wbest, int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof);
void leb_an_stats(const AnState*, double* flops_fwd, long long* ins_fwd, long long* tape_ins, int* ntasks, int* max_slots);

// ---- zonotope fold (inflate.cu)
cudaError_t leb_launch_inflate(size_t rows, int n, const float* r_lo, const float* r_hi, const float* E_diag, float pad,
                               float* c_bar, float* R_diag, float* Ebar_dense, cudaStream_t st, long long* launches,
                               LebProf* prof);
cudaError_t leb_launch_inflate_vjp(size_t count, const float* gc, const float* gR, float* g_lo, float* g_hi,
                                   cudaStream_t st, long long* launches);

// ---- disturbance error, tube propagation, J_err (tube.cu)
cudaError_t leb_launch_dist_add(size_t rows, int nw, const float* E_lo, const float* E_hi, const float* E_nom, float* r_lo,
                                float* r_hi, cudaStream_t st, long long* launches, LebProf* prof);
cudaError_t leb_launch_tube(int B, int T, int n, int N, const float* Phi, const float* c_bar, const float* R_diag,
                            const float* E_diag, float* h_mu, float* h_sigma, cudaStream_t st, long long* launches,
                            LebProf* prof);
cudaError_t leb_launch_jerr(int B, int T, int n, int N, const float* Phi, const float* R_diag, const float* E_diag,
                            float* partial, float* J, float* grad_R, cudaStream_t st, long long* launches, LebProf* prof);
cudaError_t leb_jerr_static_setup(int device);      // tube.cu: resolves the static scratch on the current device
cudaError_t leb_launch_jerr_static(int device, int B, int T, int n, int N, const float* Phi, const float* R_diag, const float* E_diag,
                                   float* J, float* grad_R, cudaStream_t st, long long* launches);

// ---- NN path (nn.cu)
struct NnState;   // packed weights + workspace, owned by the context
NnState* leb_nn_create();
void leb_nn_destroy(NnState*);
leb_status leb_nn_set_mlp(NnState*, const leb_mlp* mlp, cudaStream_t st, long long* launches);
leb_status leb_nn_set_chunk(NnState*, int tiles);
bool leb_nn_ready(const NnState*);
int leb_nn_n(const NnState*);
int leb_nn_N(const NnState*);
leb_status leb_nn_forward(NnState*, int tiles, const float* nom, const float* rad, const float* mu, const float* J, int ld_in,
                          float* r_lo, float* r_hi, float* margin, int ld_out, unsigned flags, int* domain_flag, cudaStream_t st,
                          long long* launches, LebProf* prof);
leb_status leb_nn_vjp(NnState*, int tiles, const float* nom, const float* rad, const float* mu, const float* g_lo,
                      const float* g_hi, int ld_in, int ld_out, float* grad_nom, float* grad_rad, float* grad_mu, unsigned flags,
                      int* domain_flag, cudaStream_t st, long long* launches, LebProf* prof);
leb_status leb_nn_alpha(NnState*, int tiles, const float* nom, const float* rad, int ld_in, int steps, float lr, float* r_lo,
                        float* r_hi, int ld_out, float* w0, float* wbest, unsigned flags, int* domain_flag, cudaStream_t st,
                        long long* launches, LebProf* prof);
void leb_nn_query(const NnState*, int* tiles, int* certified, int* vjp_reused);
leb_status leb_nn_get_hidden(NnState*, int layer, float* l, float* u, cudaStream_t st, long long* launches);
leb_status leb_nn_get_coeffs(NnState*, int target, float* out, cudaStream_t st, long long* launches);
leb_status leb_nn_get_jacobian(NnState*, float* out, cudaStream_t st, long long* launches);
leb_status leb_nn_get_slopes(NnState*, int layer, float* kU, float* kL, cudaStream_t st, long long* launches);

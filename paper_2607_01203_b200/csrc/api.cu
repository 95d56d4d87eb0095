// api.cu -- the extern "C" boundary declared in include/leb.h: argument validation, host-IO
// staging, dispatch to the kernels' launchers.  No numerical step of the method runs on the host.
#include <stdio.h>
#include <stdint.h>
#include <new>
#include "internal.h"

struct leb_ctx {
    int device = 0;
    AnState* an = nullptr;
    NnState* nn = nullptr;
    int* domain_flag = nullptr;     // device
    long long launches = 0;
    LebProf prof;
    // staging for LEB_FLAG_HOST_IO (grown on demand)
    float* stage[8] = {nullptr};
    size_t stage_bytes[8] = {0};
};

namespace {

struct DeviceGuard {
    int prev = 0;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline bool al4(const void* p) { return ((uintptr_t)p & 3) == 0; }

float* stage_buf(leb_ctx* c, int slot, size_t bytes) {
    if (bytes == 0) bytes = 16;
    if (c->stage_bytes[slot] < bytes) {
        if (c->stage[slot]) { cudaDeviceSynchronize(); cudaFree(c->stage[slot]); c->stage[slot] = nullptr; c->stage_bytes[slot] = 0; }
        if (cudaMalloc(&c->stage[slot], bytes) != cudaSuccess) return nullptr;
        c->stage_bytes[slot] = bytes;
    }
    return c->stage[slot];
}

// host -> staging (returns device pointer) or pass-through
const float* in_ptr(leb_ctx* c, int slot, const float* p, size_t count, bool host, cudaStream_t st, bool* ok) {
    if (!host || !p) return p;
    float* d = stage_buf(c, slot, count * sizeof(float));
    if (!d) { *ok = false; return nullptr; }
    if (cudaMemcpyAsync(d, p, count * sizeof(float), cudaMemcpyHostToDevice, st) != cudaSuccess) *ok = false;
    return d;
}
float* out_ptr(leb_ctx* c, int slot, float* p, size_t count, bool host, bool* ok) {
    if (!host || !p) return p;
    float* d = stage_buf(c, slot, count * sizeof(float));
    if (!d) *ok = false;
    return d;
}
void out_copy(float* host_p, const float* dev_p, size_t count, bool host, cudaStream_t st, bool* ok) {
    if (!host || !host_p) return;
    if (cudaMemcpyAsync(host_p, dev_p, count * sizeof(float), cudaMemcpyDeviceToHost, st) != cudaSuccess) *ok = false;
}

leb_status check_traj(int B, int T, int N, int n, int ld_in, int ld_out) {
    if (B < 0 || T < 0) return LEB_ERR_ARG;
    if ((long long)B * T > 2000000000LL) return LEB_ERR_SHAPE;
    if (ld_in < N || ld_out < n) return LEB_ERR_SHAPE;
    return LEB_OK;
}

}  // namespace

extern "C" {

const char* leb_status_str(leb_status s) {
    switch (s) {
        case LEB_OK: return "ok";
        case LEB_ERR_ARG: return "bad argument";
        case LEB_ERR_SHAPE: return "bad shape";
        case LEB_ERR_ALIGN: return "misaligned pointer";
        case LEB_ERR_DOMAIN: return "domain error in some tile";
        case LEB_ERR_UNSUPPORTED: return "unsupported";
        case LEB_ERR_CUDA: return "CUDA error";
        case LEB_ERR_NOMEM: return "out of device memory";
        case LEB_ERR_STATE: return "model not set";
        case LEB_ERR_CAPACITY: return "problem larger than the fixed capacity of this entry point";
    }
    return "unknown";
}

leb_status leb_create(leb_ctx** out, int device) {
    if (!out) return LEB_ERR_ARG;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return LEB_ERR_CUDA;
    DeviceGuard guard(device);
    leb_ctx* c = new (std::nothrow) leb_ctx();
    if (!c) return LEB_ERR_NOMEM;
    c->device = device;
    if (cudaMalloc(&c->domain_flag, sizeof(int)) != cudaSuccess) { delete c; return LEB_ERR_NOMEM; }
    cudaMemset(c->domain_flag, 0, sizeof(int));
    c->nn = leb_nn_create();
    c->an = leb_an_create();
    (void)leb_jerr_static_setup(device);      // static scratch of leb_jerr_static; a failure is reported by that entry point
    if (!c->nn || !c->an) { leb_nn_destroy(c->nn); leb_an_destroy(c->an); cudaFree(c->domain_flag); delete c; return LEB_ERR_NOMEM; }
    *out = c;
    return LEB_OK;
}

leb_status leb_destroy(leb_ctx* c) {
    if (!c) return LEB_OK;
    DeviceGuard guard(c->device);
    cudaDeviceSynchronize();
    leb_nn_destroy(c->nn);
    leb_an_destroy(c->an);
    c->prof.destroy();
    for (int i = 0; i < 8; ++i) if (c->stage[i]) cudaFree(c->stage[i]);
    if (c->domain_flag) cudaFree(c->domain_flag);
    delete c;
    return LEB_OK;
}

leb_status leb_set_analytic(leb_ctx* c, const leb_analytic_model* m) {
    if (!c || !m) return LEB_ERR_ARG;
    if (m->model_id < LEB_MODEL_UNICYCLE || m->model_id > LEB_MODEL_QUADCENTROID) return LEB_ERR_UNSUPPORTED;
    if (m->model_id != LEB_MODEL_UNICYCLE && m->integ != LEB_INTEG_EULER && m->integ != LEB_INTEG_RK4) return LEB_ERR_ARG;
    if ((m->model_id == LEB_MODEL_QUADCHAIN || m->model_id == LEB_MODEL_QUADCENTROID) && (m->n_units < 1 || m->n_units > 4096)) return LEB_ERR_SHAPE;
    if (!(m->dt > 0.f)) return LEB_ERR_ARG;
    if (m->model_id != LEB_MODEL_UNICYCLE && !(m->Jx > 0.f)) return LEB_ERR_ARG;
    if (m->model_id != LEB_MODEL_UNICYCLE && m->model_id != LEB_MODEL_SATELLITE && !(m->mass > 0.f)) return LEB_ERR_ARG;
    if (m->model_id != LEB_MODEL_UNICYCLE && m->model_id != LEB_MODEL_PLANAR_QUAD && (!(m->Jy > 0.f) || !(m->Jz > 0.f))) return LEB_ERR_ARG;
    DeviceGuard guard(c->device);
    return leb_an_set_model(c->an, leb_make_model(*m));
}

leb_status leb_set_mlp(leb_ctx* c, const leb_mlp* m, void* stream) {
    if (!c) return LEB_ERR_ARG;
    DeviceGuard guard(c->device);
    return leb_nn_set_mlp(c->nn, m, (cudaStream_t)stream, &c->launches);
}

leb_status leb_set_nn_chunk(leb_ctx* c, int tiles) {
    if (!c) return LEB_ERR_ARG;
    DeviceGuard guard(c->device);
    return leb_nn_set_chunk(c->nn, tiles);
}

leb_status leb_analytic_fwd(leb_ctx* c, int B, int T, const float* nom, const float* rad, const float* mu, int ld_in,
                            float* r_lo, float* r_hi, int ld_out, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0) return LEB_ERR_ARG;
    if (!leb_an_ready(c->an)) return LEB_ERR_STATE;
    if (B == 0 || T == 0) return LEB_OK;            // empty batch: nothing to do, pointers may be NULL
    if (!nom || !rad || !r_lo || !r_hi) return LEB_ERR_ARG;
    leb_status s = check_traj(B, T, leb_an_N(c->an), leb_an_n(c->an), ld_in, ld_out);
    if (s != LEB_OK) return s;
    if (!al4(nom) || !al4(rad) || !al4(mu) || !al4(r_lo) || !al4(r_hi)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_nom = in_ptr(c, 0, nom, tiles * ld_in, host, st, &ok);
    const float* d_rad = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    const float* d_mu = in_ptr(c, 4, mu, tiles * ld_in, host, st, &ok);
    float* d_lo = out_ptr(c, 2, r_lo, tiles * ld_out, host, &ok);
    float* d_hi = out_ptr(c, 3, r_hi, tiles * ld_out, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    s = leb_an_forward(c->an, (int)tiles, d_nom, d_rad, d_mu, ld_in, d_lo, d_hi, ld_out, c->domain_flag, st, &c->launches, &c->prof);
    if (s != LEB_OK) return s;
    out_copy(r_lo, d_lo, tiles * ld_out, host, st, &ok);
    out_copy(r_hi, d_hi, tiles * ld_out, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_analytic_partition_fwd(leb_ctx* c, int B, int T, const float* nom, const float* rad, const float* mu, int ld_in,
                                      const int* splits, float* r_lo, float* r_hi, int ld_out, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || !splits) return LEB_ERR_ARG;
    if (!leb_an_ready(c->an)) return LEB_ERR_STATE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!nom || !rad || !r_lo || !r_hi) return LEB_ERR_ARG;
    leb_status s = check_traj(B, T, leb_an_N(c->an), leb_an_n(c->an), ld_in, ld_out);
    if (s != LEB_OK) return s;
    if (!al4(nom) || !al4(rad) || !al4(mu) || !al4(r_lo) || !al4(r_hi)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_nom = in_ptr(c, 0, nom, tiles * ld_in, host, st, &ok);
    const float* d_rad = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    const float* d_mu = in_ptr(c, 4, mu, tiles * ld_in, host, st, &ok);
    float* d_lo = out_ptr(c, 2, r_lo, tiles * ld_out, host, &ok);
    float* d_hi = out_ptr(c, 3, r_hi, tiles * ld_out, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    s = leb_an_partition(c->an, (int)tiles, d_nom, d_rad, d_mu, ld_in, splits, d_lo, d_hi, ld_out, c->domain_flag, st, &c->launches, &c->prof);
    if (s != LEB_OK) return s;
    out_copy(r_lo, d_lo, tiles * ld_out, host, st, &ok);
    out_copy(r_hi, d_hi, tiles * ld_out, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_analytic_partition_vjp(leb_ctx* c, int B, int T, const float* nom, const float* rad, const float* mu, int ld_in,
                                      const int* splits, const float* g_lo, const float* g_hi, int ld_out, float* grad_nom,
                                      float* grad_rad, float* grad_mu, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || !splits) return LEB_ERR_ARG;
    if (!leb_an_ready(c->an)) return LEB_ERR_STATE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!nom || !rad || !g_lo || !g_hi || !grad_nom || !grad_rad || (mu && !grad_mu)) return LEB_ERR_ARG;
    leb_status s = check_traj(B, T, leb_an_N(c->an), leb_an_n(c->an), ld_in, ld_out);
    if (s != LEB_OK) return s;
    if (!al4(nom) || !al4(rad) || !al4(mu) || !al4(g_lo) || !al4(g_hi) || !al4(grad_nom) || !al4(grad_rad) || !al4(grad_mu)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_nom = in_ptr(c, 0, nom, tiles * ld_in, host, st, &ok);
    const float* d_rad = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    const float* d_glo = in_ptr(c, 2, g_lo, tiles * ld_out, host, st, &ok);
    const float* d_ghi = in_ptr(c, 3, g_hi, tiles * ld_out, host, st, &ok);
    const float* d_mu = in_ptr(c, 4, mu, tiles * ld_in, host, st, &ok);
    float* d_gn = out_ptr(c, 6, grad_nom, tiles * ld_in, host, &ok);
    float* d_gr = out_ptr(c, 7, grad_rad, tiles * ld_in, host, &ok);
    float* d_gm = out_ptr(c, 5, (mu ? grad_mu : nullptr), tiles * ld_in, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    s = leb_an_partition_vjp(c->an, (int)tiles, d_nom, d_rad, d_mu, ld_in, splits, d_glo, d_ghi, ld_out, d_gn, d_gr, d_gm, c->domain_flag, st,
                             &c->launches, &c->prof);
    if (s != LEB_OK) return s;
    out_copy(grad_nom, d_gn, tiles * ld_in, host, st, &ok);
    out_copy(grad_rad, d_gr, tiles * ld_in, host, st, &ok);
    if (mu) out_copy(grad_mu, d_gm, tiles * ld_in, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_analytic_pgd(leb_ctx* c, int B, int T, const float* centre, const float* rad, const float* eps, int ld_in, int steps,
                            float lr, float* nom, float* width0, float* width, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || steps < 0 || !(lr >= 0.f)) return LEB_ERR_ARG;
    if (!leb_an_ready(c->an)) return LEB_ERR_STATE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!centre || !rad || !eps || !nom || !width0 || !width) return LEB_ERR_ARG;
    if (ld_in < leb_an_N(c->an)) return LEB_ERR_SHAPE;
    if (!al4(centre) || !al4(rad) || !al4(eps) || !al4(nom) || !al4(width0) || !al4(width)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_c = in_ptr(c, 0, centre, tiles * ld_in, host, st, &ok);
    const float* d_r = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    const float* d_e = in_ptr(c, 4, eps, tiles * ld_in, host, st, &ok);
    float* d_n = const_cast<float*>(in_ptr(c, 2, nom, tiles * ld_in, host, st, &ok));
    float* d_w0 = out_ptr(c, 6, width0, tiles, host, &ok);
    float* d_w = out_ptr(c, 7, width, tiles, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    leb_status s = leb_an_pgd(c->an, (int)tiles, d_c, d_r, d_e, ld_in, steps, lr, d_n, d_w0, d_w, c->domain_flag, st, &c->launches, &c->prof);
    if (s != LEB_OK) return s;
    out_copy(nom, d_n, tiles * ld_in, host, st, &ok);
    out_copy(width0, d_w0, tiles, host, st, &ok);
    out_copy(width, d_w, tiles, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_nn_fwd(leb_ctx* c, int B, int T, const float* nom, const float* rad, const float* mu, const float* J, int ld_in,
                      float* r_lo, float* r_hi, float* margin, int ld_out, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!nom || !rad || !r_lo || !r_hi) return LEB_ERR_ARG;
    const int n = leb_nn_n(c->nn), N = leb_nn_N(c->nn);
    leb_status s = check_traj(B, T, N, n, ld_in, ld_out);
    if (s != LEB_OK) return s;
    if (!al4(nom) || !al4(rad) || !al4(mu) || !al4(r_lo) || !al4(r_hi) || !al4(J) || !al4(margin)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_nom = in_ptr(c, 0, nom, tiles * ld_in, host, st, &ok);
    const float* d_rad = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    const float* d_J = in_ptr(c, 4, J, tiles * (size_t)n * N, host, st, &ok);
    const float* d_mu = in_ptr(c, 6, mu, tiles * ld_in, host, st, &ok);
    float* d_lo = out_ptr(c, 2, r_lo, tiles * ld_out, host, &ok);
    float* d_hi = out_ptr(c, 3, r_hi, tiles * ld_out, host, &ok);
    float* d_mg = out_ptr(c, 5, margin, tiles * ld_out, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    s = leb_nn_forward(c->nn, (int)tiles, d_nom, d_rad, d_mu, d_J, ld_in, d_lo, d_hi, d_mg, ld_out, flags, c->domain_flag, st, &c->launches, &c->prof);
    if (s != LEB_OK) return s;
    out_copy(r_lo, d_lo, tiles * ld_out, host, st, &ok);
    out_copy(r_hi, d_hi, tiles * ld_out, host, st, &ok);
    out_copy(margin, d_mg, tiles * ld_out, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_nn_alpha_fwd(leb_ctx* c, int B, int T, const float* nom, const float* rad, int ld_in, int steps, float lr, float* r_lo,
                            float* r_hi, int ld_out, float* width0, float* width, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || steps < 0 || !(lr >= 0.f)) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!nom || !rad || !r_lo || !r_hi || !width0 || !width) return LEB_ERR_ARG;
    const int n = leb_nn_n(c->nn), N = leb_nn_N(c->nn);
    leb_status s = check_traj(B, T, N, n, ld_in, ld_out);
    if (s != LEB_OK) return s;
    if (!al4(nom) || !al4(rad) || !al4(r_lo) || !al4(r_hi) || !al4(width0) || !al4(width)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_nom = in_ptr(c, 0, nom, tiles * ld_in, host, st, &ok);
    const float* d_rad = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    float* d_lo = out_ptr(c, 2, r_lo, tiles * ld_out, host, &ok);
    float* d_hi = out_ptr(c, 3, r_hi, tiles * ld_out, host, &ok);
    float* d_w0 = out_ptr(c, 6, width0, tiles, host, &ok);
    float* d_w = out_ptr(c, 7, width, tiles, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    s = leb_nn_alpha(c->nn, (int)tiles, d_nom, d_rad, ld_in, steps, lr, d_lo, d_hi, ld_out, d_w0, d_w, flags, c->domain_flag, st, &c->launches, &c->prof);
    if (s != LEB_OK) return s;
    out_copy(r_lo, d_lo, tiles * ld_out, host, st, &ok);
    out_copy(r_hi, d_hi, tiles * ld_out, host, st, &ok);
    out_copy(width0, d_w0, tiles, host, st, &ok);
    out_copy(width, d_w, tiles, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_vjp_mu(leb_ctx* c, int kind, int B, int T, const float* nom, const float* rad, const float* mu, const float* g_lo,
                      const float* g_hi, int ld_in, int ld_out, float* grad_nom, float* grad_rad, float* grad_mu, unsigned flags,
                      void* stream) {
    if (!c || B < 0 || T < 0) return LEB_ERR_ARG;
    if (kind != 0 && kind != 1) return LEB_ERR_ARG;
    if ((B == 0 || T == 0) && (kind == 0 ? leb_an_ready(c->an) : leb_nn_ready(c->nn))) return LEB_OK;
    if (!nom || !rad || !g_lo || !g_hi || !grad_nom || !grad_rad) return LEB_ERR_ARG;
    int n, N;
    if (kind == 0) {
        if (!leb_an_ready(c->an)) return LEB_ERR_STATE;
        n = leb_an_n(c->an); N = leb_an_N(c->an);
    } else {
        if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
        n = leb_nn_n(c->nn); N = leb_nn_N(c->nn);
    }
    leb_status s = check_traj(B, T, N, n, ld_in, ld_out);
    if (s != LEB_OK) return s;
    if (!al4(nom) || !al4(rad) || !al4(mu) || !al4(g_lo) || !al4(g_hi) || !al4(grad_nom) || !al4(grad_rad) || !al4(grad_mu)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t tiles = (size_t)B * T;
    bool ok = true;
    const float* d_nom = in_ptr(c, 0, nom, tiles * ld_in, host, st, &ok);
    const float* d_rad = in_ptr(c, 1, rad, tiles * ld_in, host, st, &ok);
    const float* d_glo = in_ptr(c, 2, g_lo, tiles * ld_out, host, st, &ok);
    const float* d_ghi = in_ptr(c, 3, g_hi, tiles * ld_out, host, st, &ok);
    const float* d_mu = in_ptr(c, 4, mu, tiles * ld_in, host, st, &ok);
    float* d_gn = out_ptr(c, 6, grad_nom, tiles * ld_in, host, &ok);
    float* d_gr = out_ptr(c, 7, grad_rad, tiles * ld_in, host, &ok);
    float* d_gm = out_ptr(c, 5, (mu ? grad_mu : nullptr), tiles * ld_in, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    if (kind == 0) {
        s = leb_an_vjp(c->an, (int)tiles, d_nom, d_rad, d_mu, d_glo, d_ghi, ld_in, ld_out, d_gn, d_gr, d_gm, c->domain_flag, st,
                       &c->launches, &c->prof);
        if (s != LEB_OK) return s;
    } else {
        s = leb_nn_vjp(c->nn, (int)tiles, d_nom, d_rad, d_mu, d_glo, d_ghi, ld_in, ld_out, d_gn, d_gr, d_gm, flags, c->domain_flag, st, &c->launches, &c->prof);
        if (s != LEB_OK) return s;
    }
    out_copy(grad_nom, d_gn, tiles * ld_in, host, st, &ok);
    out_copy(grad_rad, d_gr, tiles * ld_in, host, st, &ok);
    if (mu) out_copy(grad_mu, d_gm, tiles * ld_in, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_vjp(leb_ctx* c, int kind, int B, int T, const float* nom, const float* rad, const float* g_lo, const float* g_hi,
                   int ld_in, int ld_out, float* grad_nom, float* grad_rad, unsigned flags, void* stream) {
    return leb_vjp_mu(c, kind, B, T, nom, rad, nullptr, g_lo, g_hi, ld_in, ld_out, grad_nom, grad_rad, nullptr, flags, stream);
}

leb_status leb_zonotope_inflate(leb_ctx* c, int B, int T, int n, const float* r_lo, const float* r_hi, const float* E_diag,
                                float pad, float* c_bar, float* R_diag, float* Ebar_dense, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || n < 1 || !(pad >= 0.f)) return LEB_ERR_ARG;
    if (B == 0 || T == 0) return LEB_OK;
    if (!r_lo || !r_hi || !c_bar || !R_diag) return LEB_ERR_ARG;
    if (!al4(r_lo) || !al4(r_hi) || !al4(c_bar) || !al4(R_diag) || !al4(Ebar_dense) || !al4(E_diag)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t rows = (size_t)B * T * n;
    bool ok = true;
    const float* d_lo = in_ptr(c, 0, r_lo, rows, host, st, &ok);
    const float* d_hi = in_ptr(c, 1, r_hi, rows, host, st, &ok);
    const float* d_E = in_ptr(c, 4, E_diag, n, host, st, &ok);
    float* d_c = out_ptr(c, 2, c_bar, rows, host, &ok);
    float* d_R = out_ptr(c, 3, R_diag, rows, host, &ok);
    float* d_Eb = out_ptr(c, 5, Ebar_dense, rows * 2 * n, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    if (leb_launch_inflate(rows, n, d_lo, d_hi, d_E, pad, d_c, d_R, d_Eb, st, &c->launches, &c->prof) != cudaSuccess) return LEB_ERR_CUDA;
    out_copy(c_bar, d_c, rows, host, st, &ok);
    out_copy(R_diag, d_R, rows, host, st, &ok);
    out_copy(Ebar_dense, d_Eb, rows * 2 * n, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_zonotope_inflate_vjp(leb_ctx* c, int B, int T, int n, const float* gc, const float* gR, float* g_lo, float* g_hi,
                                    unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || n < 1) return LEB_ERR_ARG;
    if (B == 0 || T == 0) return LEB_OK;
    if (!gc || !gR || !g_lo || !g_hi) return LEB_ERR_ARG;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t count = (size_t)B * T * n;
    bool ok = true;
    const float* d_gc = in_ptr(c, 0, gc, count, host, st, &ok);
    const float* d_gR = in_ptr(c, 1, gR, count, host, st, &ok);
    float* d_lo = out_ptr(c, 2, g_lo, count, host, &ok);
    float* d_hi = out_ptr(c, 3, g_hi, count, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    if (leb_launch_inflate_vjp(count, d_gc, d_gR, d_lo, d_hi, st, &c->launches) != cudaSuccess) return LEB_ERR_CUDA;
    out_copy(g_lo, d_lo, count, host, st, &ok);
    out_copy(g_hi, d_hi, count, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_dist_add(leb_ctx* c, int B, int T, int n, int nw, const float* E_lo, const float* E_hi, const float* E_nom,
                        float* r_lo, float* r_hi, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || n < 1 || nw < 1) return LEB_ERR_ARG;
    if (B == 0 || T == 0) return LEB_OK;
    if (!E_lo || !E_hi || !E_nom || !r_lo || !r_hi) return LEB_ERR_ARG;
    if (!al4(E_lo) || !al4(E_hi) || !al4(E_nom) || !al4(r_lo) || !al4(r_hi)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const size_t rows = (size_t)B * T * n;
    bool ok = true;
    const float* d_a = in_ptr(c, 0, E_lo, rows * nw, host, st, &ok);
    const float* d_b = in_ptr(c, 1, E_hi, rows * nw, host, st, &ok);
    const float* d_c = in_ptr(c, 4, E_nom, rows * nw, host, st, &ok);
    float* d_lo = const_cast<float*>(in_ptr(c, 2, r_lo, rows, host, st, &ok));
    float* d_hi = const_cast<float*>(in_ptr(c, 3, r_hi, rows, host, st, &ok));
    if (!ok) return LEB_ERR_NOMEM;
    if (leb_launch_dist_add(rows, nw, d_a, d_b, d_c, d_lo, d_hi, st, &c->launches, &c->prof) != cudaSuccess) return LEB_ERR_CUDA;
    out_copy(r_lo, d_lo, rows, host, st, &ok);
    out_copy(r_hi, d_hi, rows, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_tube_propagate(leb_ctx* c, int B, int T, int n, int m, const float* Phi, const float* c_bar, const float* R_diag,
                              const float* E_diag, float* h_mu, float* h_sigma, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || n < 1 || m < 0) return LEB_ERR_ARG;
    if (n > 8192) return LEB_ERR_UNSUPPORTED;
    if (T > 65535 || B > 65535) return LEB_ERR_SHAPE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!Phi || !c_bar || !R_diag || !h_mu || !h_sigma) return LEB_ERR_ARG;
    if (((uintptr_t)Phi & 15) || !al4(c_bar) || !al4(R_diag) || !al4(E_diag) || !al4(h_mu) || !al4(h_sigma)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const int N = n + m;
    const size_t nphi = (size_t)B * ((size_t)T * (T + 1) / 2) * N * n, nv = (size_t)B * T * n, no = (size_t)B * T * N;
    bool ok = true;
    const float* d_P = in_ptr(c, 0, Phi, nphi, host, st, &ok);
    const float* d_c = in_ptr(c, 1, c_bar, nv, host, st, &ok);
    const float* d_R = in_ptr(c, 2, R_diag, nv, host, st, &ok);
    const float* d_E = in_ptr(c, 4, E_diag, n, host, st, &ok);
    float* d_m = out_ptr(c, 6, h_mu, no, host, &ok);
    float* d_s = out_ptr(c, 7, h_sigma, no, host, &ok);
    if (!ok) return LEB_ERR_NOMEM;
    if (leb_launch_tube(B, T, n, N, d_P, d_c, d_R, d_E, d_m, d_s, st, &c->launches, &c->prof) != cudaSuccess) return LEB_ERR_CUDA;
    out_copy(h_mu, d_m, no, host, st, &ok);
    out_copy(h_sigma, d_s, no, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_jerr(leb_ctx* c, int B, int T, int n, int m, const float* Phi, const float* R_diag, const float* E_diag,
                    float* J_err, float* grad_R, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || n < 1 || m < 0) return LEB_ERR_ARG;
    if (n > 1024) return LEB_ERR_UNSUPPORTED;
    if (T > 65535 || B > 65535) return LEB_ERR_SHAPE;
    if (B == 0 || T == 0) return LEB_OK;
    if (!Phi || !R_diag || !J_err) return LEB_ERR_ARG;
    if (!al4(Phi) || !al4(R_diag) || !al4(E_diag) || !al4(J_err) || !al4(grad_R)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool host = flags & LEB_FLAG_HOST_IO;
    const int N = n + m;
    const size_t nphi = (size_t)B * ((size_t)T * (T + 1) / 2) * N * n, nv = (size_t)B * T * n;
    bool ok = true;
    const float* d_P = in_ptr(c, 0, Phi, nphi, host, st, &ok);
    const float* d_R = in_ptr(c, 2, R_diag, nv, host, st, &ok);
    const float* d_E = in_ptr(c, 4, E_diag, n, host, st, &ok);
    float* d_J = out_ptr(c, 6, J_err, (size_t)B, host, &ok);
    float* d_g = out_ptr(c, 7, grad_R, nv, host, &ok);
    float* d_part = stage_buf(c, 5, (size_t)B * T * sizeof(float));
    if (!ok || !d_part) return LEB_ERR_NOMEM;
    if (leb_launch_jerr(B, T, n, N, d_P, d_R, d_E, d_part, d_J, d_g, st, &c->launches, &c->prof) != cudaSuccess) return LEB_ERR_CUDA;
    out_copy(J_err, d_J, (size_t)B, host, st, &ok);
    out_copy(grad_R, d_g, nv, host, st, &ok);
    return ok ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_jerr_static(leb_ctx* c, int B, int T, int n, int m, const float* Phi, const float* R_diag, const float* E_diag,
                           float* J_err, float* grad_R, unsigned flags, void* stream) {
    if (!c || B < 0 || T < 0 || n < 1 || m < 0) return LEB_ERR_ARG;
    if (flags & LEB_FLAG_HOST_IO) return LEB_ERR_ARG;                 // staging host buffers would allocate
    if (n > 1024) return LEB_ERR_UNSUPPORTED;
    if (T > 65535 || B > 65535) return LEB_ERR_SHAPE;
    if ((long long)B * T > (long long)LEB_JERR_STATIC_MAX) return LEB_ERR_CAPACITY;
    if (B == 0 || T == 0) return LEB_OK;
    if (!Phi || !R_diag || !J_err) return LEB_ERR_ARG;
    if (!al4(Phi) || !al4(R_diag) || !al4(E_diag) || !al4(J_err) || !al4(grad_R)) return LEB_ERR_ALIGN;
    DeviceGuard guard(c->device);
    const cudaError_t e = leb_launch_jerr_static(c->device, B, T, n, n + m, Phi, R_diag, E_diag, J_err, grad_R, (cudaStream_t)stream, &c->launches);
    return e == cudaSuccess ? LEB_OK : LEB_ERR_CUDA;
}

leb_status leb_domain_flag(leb_ctx* c, int* flag, void* stream) {
    if (!c || !flag) return LEB_ERR_ARG;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    int h = 0;
    if (cudaMemcpyAsync(&h, c->domain_flag, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess) return LEB_ERR_CUDA;
    if (cudaMemsetAsync(c->domain_flag, 0, sizeof(int), st) != cudaSuccess) return LEB_ERR_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return LEB_ERR_CUDA;
    *flag = h;
    return LEB_OK;
}

leb_status leb_nn_hidden_bounds(leb_ctx* c, int layer, float* l, float* u, void* stream) {
    if (!c || !l || !u) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    DeviceGuard guard(c->device);
    return leb_nn_get_hidden(c->nn, layer, l, u, (cudaStream_t)stream, &c->launches);
}

leb_status leb_nn_chain_coeffs(leb_ctx* c, int target, float* out, void* stream) {
    if (!c || !out) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    DeviceGuard guard(c->device);
    return leb_nn_get_coeffs(c->nn, target, out, (cudaStream_t)stream, &c->launches);
}

leb_status leb_nn_slopes(leb_ctx* c, int layer, float* kU, float* kL, void* stream) {
    if (!c || !kU || !kL) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    DeviceGuard guard(c->device);
    return leb_nn_get_slopes(c->nn, layer, kU, kL, (cudaStream_t)stream, &c->launches);
}

leb_status leb_nn_jacobian(leb_ctx* c, float* out, void* stream) {
    if (!c || !out) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    DeviceGuard guard(c->device);
    return leb_nn_get_jacobian(c->nn, out, (cudaStream_t)stream, &c->launches);
}

leb_status leb_nn_state(leb_ctx* c, int* tiles, int* certified, int* vjp_reused) {
    if (!c || !tiles || !certified || !vjp_reused) return LEB_ERR_ARG;
    if (!leb_nn_ready(c->nn)) return LEB_ERR_STATE;
    leb_nn_query(c->nn, tiles, certified, vjp_reused);
    return LEB_OK;
}

leb_status leb_analytic_tape_stats(leb_ctx* c, double* flops_per_tile, long long* ins_per_tile, long long* tape_ins, int* tasks,
                                   int* max_slots) {
    if (!c || !flops_per_tile || !ins_per_tile || !tape_ins || !tasks || !max_slots) return LEB_ERR_ARG;
    if (!leb_an_ready(c->an)) return LEB_ERR_STATE;
    leb_an_stats(c->an, flops_per_tile, ins_per_tile, tape_ins, tasks, max_slots);
    return LEB_OK;
}

long long leb_launch_count(const leb_ctx* c) { return c ? c->launches : 0; }

leb_status leb_profile(leb_ctx* c, int enable) {
    if (!c) return LEB_ERR_ARG;
    c->prof.on = enable != 0;
    return LEB_OK;
}

leb_status leb_profile_read(leb_ctx* c, int kernel_class, double* ms, double* work, long long* launches, void* stream) {
    if (!c || !ms || !work || !launches) return LEB_ERR_ARG;
    if (kernel_class < 0 || kernel_class >= LEB_KC_COUNT) return LEB_ERR_ARG;
    DeviceGuard guard(c->device);
    if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return LEB_ERR_CUDA;
    double total = 0.0;
    for (size_t i = 0; i < c->prof.used; ++i) {
        if (c->prof.recs[i].kc != kernel_class) continue;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, c->prof.recs[i].a, c->prof.recs[i].b) != cudaSuccess) return LEB_ERR_CUDA;
        total += t;
    }
    *ms = total;
    *work = c->prof.work[kernel_class];
    *launches = c->prof.count[kernel_class];
    return LEB_OK;
}

leb_status leb_profile_reset(leb_ctx* c) {
    if (!c) return LEB_ERR_ARG;
    c->prof.used = 0;
    for (int k = 0; k < LEB_KC_COUNT; ++k) { c->prof.work[k] = 0.0; c->prof.count[k] = 0; }
    return LEB_OK;
}

}  // extern "C"

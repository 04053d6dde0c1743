// nmf_api.cu -- the extern "C" boundary declared in include/nmf.h:
// argument validation, plan/workspace management, dispatch to the kernel families.
#include "nmf_common.cuh"
#include <new>

namespace {

inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

size_t plan_workspace(nmf_plan* p) {
    size_t g = nmf_generic_workspace(p);
    size_t f = nmf_fused_workspace(p);
    size_t t = nmf_tc_workspace(p);
    size_t ts = nmf_tcsplit_workspace(p);
    if (ts > t) t = ts;
    size_t st = nmf_stream_workspace(p);
    if (st > t) t = st;
    size_t rs = nmf_resident_workspace(p);
    if (rs > t) t = rs;
    size_t sel = nmf_select_workspace(p);
    if (f > g) g = f;
    if (t > g) g = t;
    if (sel > g) g = sel;
    size_t main = nmf_align_up(g, 256);
    return main + nmf_align_up(nmf_aux_workspace(p), 256);
}

// every call must run with the plan's device current (launches, function attributes and copies use the current device)
int check_device(const nmf_plan* p) {
    int d = -1;
    if (cudaGetDevice(&d) != cudaSuccess) return NMF_ERR_CUDA;
    return d == p->device ? NMF_OK : NMF_ERR_INVALID_ARG;
}

int check_ws(const nmf_plan* p) {
    int rc = check_device(p);
    if (rc) return rc;
    if (!p->ws || p->ws_bytes < p->ws_needed) return NMF_ERR_WORKSPACE;
    return NMF_OK;
}

// 0 auto: split tensor core (K <= 128; the fastest family on every measured shape but the smallest) > fused tensor core
// (K <= 64) > fused FFMA > generic.  Problems of at most 64 pixel tiles in all (tiny: 32) are launch-bound: there the
// fused FFMA kernel (one light kernel + the update per iteration: 9.5 us against 13.6 us at tiny) comes first.  With
// K <= 8 the streaming FP32 kernel (X, Omega once over HBM, no BF16 split) is faster than the tensor-core kernels.
int pick_variant(const nmf_plan* p) {
    if (p->variant_req == 1) return 1;
    if (p->variant_req == 5) return nmf_stream_available(p) ? 5 : 1;
    if (p->variant_req == 6) return nmf_resident_available(p) ? 6 : 1;
    if (p->variant_req == 0 && nmf_resident_available(p)) return 6;    // small enough to stay on chip: one launch per fit
    if (p->variant_req == 2) return nmf_fused_available(p) ? 2 : 1;
    if (p->variant_req == 3) return nmf_tc_available(p) ? 3 : 1;
    if (p->variant_req == 0 && nmf_fused_available(p) && (p->P + 127) / 128 * p->batch <= 64) return 2;
    if (p->variant_req == 0 && nmf_stream_available(p)) return 5;
    if (nmf_tcsplit_available(p)) return 4;
    if (p->variant_req == 4) return 1;
    if (nmf_tc_available(p)) return 3;
    return nmf_fused_available(p) ? 2 : 1;
}

int fit_common(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters, int batch) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!X || !Om || !W || !H || iters < 0 || batch < 1 || batch > p->batch) return NMF_ERR_INVALID_ARG;
    if (misaligned(X) || misaligned(Om) || misaligned(W) || misaligned(H)) return NMF_ERR_ALIGNMENT;
    int rc = check_ws(p);
    if (rc) return rc;
    if (iters == 0) return NMF_OK;
    if (p->variant_req == 2 && !nmf_fused_available(p)) return NMF_ERR_UNSUPPORTED;
    if (p->variant_req == 3 && !nmf_tc_available(p)) return NMF_ERR_UNSUPPORTED;
    if (p->variant_req == 4 && !nmf_tcsplit_available(p)) return NMF_ERR_UNSUPPORTED;
    if (p->variant_req == 5 && !nmf_stream_available(p)) return NMF_ERR_UNSUPPORTED;
    if (p->variant_req == 6 && !nmf_resident_available(p)) return NMF_ERR_UNSUPPORTED;
    const int v = pick_variant(p);
    if (v == 6) return nmf_resident_fit(p, X, Om, W, H, iters);
    if (v == 5) return nmf_stream_fit(p, X, Om, W, H, iters, batch);
    if (v == 4) return nmf_tcsplit_fit(p, X, Om, W, H, iters, batch);
    if (v == 3) return nmf_tc_fit(p, X, Om, W, H, iters, batch);
    if (v == 2) return nmf_fused_fit(p, X, Om, W, H, iters, batch);
    return nmf_generic_fit(p, X, Om, W, H, iters, batch);
}

int ensure_stage(nmf_plan* p, size_t bytes) {
    if (p->stage_bytes >= bytes) return NMF_OK;
    if (p->stage_user) return NMF_ERR_WORKSPACE;         // a caller-provided staging buffer is never replaced behind the caller
    if (p->stage) { cudaFree(p->stage); p->stage = nullptr; p->stage_bytes = 0; }
    NMF_CUDA_TRY(p, cudaMalloc(&p->stage, bytes));
    p->stage_bytes = bytes;
    return NMF_OK;
}

int ensure_own_ws(nmf_plan* p) {
    if (p->ws && p->ws_bytes >= p->ws_needed) return NMF_OK;
    if (!p->own_ws) NMF_CUDA_TRY(p, cudaMalloc(&p->own_ws, p->ws_needed));
    p->ws = p->own_ws; p->ws_bytes = p->ws_needed;
    return NMF_OK;
}

}  // namespace

extern "C" {

int nmf_plan_create(nmf_plan** out, int N, long long P, int K, int batch, int max_targets) {
    if (!out) return NMF_ERR_INVALID_ARG;
    *out = nullptr;
    if (N < 1 || P < 1 || K < 1 || batch < 1 || max_targets < 0) return NMF_ERR_INVALID_ARG;
    if (P % 4 != 0) return NMF_ERR_ALIGNMENT;
    if (N > NMF_MAX_N || K > NMF_MAX_K || max_targets > 4096) return NMF_ERR_UNSUPPORTED;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return NMF_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return NMF_ERR_CUDA;
    if (prop.major != 10) return NMF_ERR_ARCH;
    if (dev < 0 || dev >= NMF_MAX_DEVICES) return NMF_ERR_UNSUPPORTED;
    nmf_plan* p = new (std::nothrow) nmf_plan();
    if (!p) return NMF_ERR_INVALID_ARG;
    if (cudaMallocHost(reinterpret_cast<void**>(&p->host_scratch), 8 * sizeof(double)) != cudaSuccess) {
        delete p;
        return NMF_ERR_CUDA;
    }
    p->N = N; p->P = P; p->K = K; p->batch = batch; p->max_targets = max_targets;
    p->device = dev; p->num_sms = prop.multiProcessorCount;
    nmf_generic_configure(p);
    nmf_fused_configure(p);
    nmf_tc_configure(p);
    nmf_tcsplit_configure(p);
    nmf_stream_configure(p);
    nmf_resident_configure(p);
    p->ws_needed = plan_workspace(p);
    *out = p;
    return NMF_OK;
}

size_t nmf_plan_workspace_bytes(const nmf_plan* p) { return p ? p->ws_needed : 0; }

int nmf_plan_set_workspace(nmf_plan* p, void* ws, size_t bytes) {
    if (!p || !ws) return NMF_ERR_INVALID_ARG;
    if (misaligned(ws)) return NMF_ERR_ALIGNMENT;
    if (bytes < p->ws_needed) return NMF_ERR_WORKSPACE;
    p->ws = ws; p->ws_bytes = bytes;
    return NMF_OK;
}

size_t nmf_plan_staging_bytes(const nmf_plan* p, int M) {
    if (!p || M < 0) return 0;
    const size_t np = nmf_align_up(sizeof(float) * (size_t)p->N * p->P, 256);
    const size_t nk = nmf_align_up(sizeof(float) * (size_t)p->N * p->K, 256);
    const size_t kp = nmf_align_up(sizeof(float) * (size_t)p->K * p->P, 256);
    const size_t mp = nmf_align_up(sizeof(float) * (size_t)M * p->P, 256);
    const size_t mk = nmf_align_up(sizeof(float) * (size_t)M * p->K, 256);
    const size_t fit = 2 * np + nk + kp, proj = 3 * mp + mk;
    return fit > proj ? fit : proj;
}

int nmf_plan_set_staging(nmf_plan* p, void* staging_dev, size_t bytes) {
    if (!p || (staging_dev == nullptr) != (bytes == 0)) return NMF_ERR_INVALID_ARG;
    if (staging_dev && misaligned(staging_dev)) return NMF_ERR_ALIGNMENT;
    if (p->stage && !p->stage_user) cudaFree(p->stage);
    p->stage = staging_dev; p->stage_bytes = bytes; p->stage_user = staging_dev != nullptr;
    return NMF_OK;
}

int nmf_plan_set_stream(nmf_plan* p, void* s) {
    if (!p) return NMF_ERR_INVALID_ARG;
    p->stream = static_cast<cudaStream_t>(s);
    return NMF_OK;
}

int nmf_plan_set_variant(nmf_plan* p, int v) {
    if (!p || v < 0 || v > 6) return NMF_ERR_INVALID_ARG;
    p->variant_req = v;
    return NMF_OK;
}

int nmf_plan_get_variant(const nmf_plan* p) {
    if (!p) return NMF_ERR_INVALID_ARG;
    return pick_variant(p);
}

int nmf_plan_destroy(nmf_plan* p) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->stage && !p->stage_user) cudaFree(p->stage);
    if (p->own_ws) cudaFree(p->own_ws);
    if (p->host_scratch) cudaFreeHost(p->host_scratch);
    if (p->g_exec) cudaGraphExecDestroy(p->g_exec);
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    delete p;
    return NMF_OK;
}

int nmf_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters) {
    return fit_common(p, X, Om, W, H, iters, 1);
}

int nmf_fit_batched(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters) {
    if (!p) return NMF_ERR_INVALID_ARG;
    return fit_common(p, X, Om, W, H, iters, p->batch);
}

int nmf_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C, int M, int iters) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!H || !T || !C || M < 1 || M > p->max_targets || iters < 0) return NMF_ERR_INVALID_ARG;
    if (misaligned(H) || misaligned(T) || misaligned(C) || (om && misaligned(om))) return NMF_ERR_ALIGNMENT;
    int rc = check_ws(p);
    if (rc) return rc;
    if (iters == 0) return NMF_OK;
    // tensor-core W phase with H fixed when the plan's fit runs there too (omega == NULL: generic path)
    if (om && pick_variant(p) == 3) return nmf_tc_project(p, H, T, om, C, M, iters);
    if (om && (pick_variant(p) == 4 || (pick_variant(p) >= 5 && nmf_tcsplit_available(p))))   // (families 5 and 6 are fit-only)
        return nmf_tcsplit_project(p, H, T, om, C, M, iters);
    return nmf_generic_project(p, H, T, om, C, M, iters);
}

int nmf_subtract(nmf_plan* p, const float* H, const float* T, const float* C, const float* om,
                 const float* factor, float fill, float* out, int M) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!H || !T || !C || !out || M < 1 || M > p->max_targets) return NMF_ERR_INVALID_ARG;
    if (out == T || out == H) return NMF_ERR_INVALID_ARG;
    if (misaligned(H) || misaligned(T) || misaligned(C) || misaligned(out) || (om && misaligned(om)))
        return NMF_ERR_ALIGNMENT;
    int rc = check_device(p);
    if (rc) return rc;
    return nmf_aux_subtract(p, H, T, C, om, factor, fill, out, M);
}

int nmf_objective(nmf_plan* p, const float* X, const float* Om, const float* W, const float* H,
                  double* out_host) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!X || !Om || !W || !H || !out_host) return NMF_ERR_INVALID_ARG;
    if (misaligned(X) || misaligned(Om) || misaligned(W) || misaligned(H)) return NMF_ERR_ALIGNMENT;
    int rc = check_ws(p);
    if (rc) return rc;
    return nmf_aux_objective(p, X, Om, W, H, out_host);
}

int nmf_fit_tol(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int max_iters, int check_every,
                double tol, int* iters_done, double* f_last) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!X || !Om || !W || !H || !iters_done || max_iters < 0 || check_every < 1 || !(tol >= 0.0)) return NMF_ERR_INVALID_ARG;
    if (misaligned(X) || misaligned(Om) || misaligned(W) || misaligned(H)) return NMF_ERR_ALIGNMENT;
    int rc = check_ws(p);
    if (rc) return rc;
    return nmf_aux_fit_tol(p, nmf_fit, X, Om, W, H, max_iters, check_every, tol, iters_done, f_last);
}

int nmf_derotate_stack(nmf_plan* p, const float* resid, const float* om, const float* angle_deg, int ny, int nx,
                       float fill, float* out, int* count, int M) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!resid || !angle_deg || !out || M < 1 || ny < 1 || nx < 1 || (long long)ny * nx != p->P) return NMF_ERR_INVALID_ARG;
    if (out == resid) return NMF_ERR_INVALID_ARG;
    if (misaligned(resid) || misaligned(out) || (om && misaligned(om))) return NMF_ERR_ALIGNMENT;
    int rc = check_device(p);
    if (rc) return rc;
    return nmf_aux_derotate_stack(p, resid, om, angle_deg, ny, nx, fill, out, count, M);
}

int nmf_fit_host(nmf_plan* p, const float* Xh, const float* Oh, float* Wh, float* Hh, int iters) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!Xh || !Oh || !Wh || !Hh || iters < 0) return NMF_ERR_INVALID_ARG;
    if (int rcd = check_device(p)) return rcd;
    const size_t np = nmf_align_up(sizeof(float) * (size_t)p->N * p->P, 256);
    const size_t nk = nmf_align_up(sizeof(float) * (size_t)p->N * p->K, 256);
    const size_t kp = nmf_align_up(sizeof(float) * (size_t)p->K * p->P, 256);
    int rc = ensure_stage(p, 2 * np + nk + kp);
    if (rc) return rc;
    rc = ensure_own_ws(p);
    if (rc) return rc;
    char* base = static_cast<char*>(p->stage);
    float* X = reinterpret_cast<float*>(base);
    float* Om = reinterpret_cast<float*>(base + np);
    float* W = reinterpret_cast<float*>(base + 2 * np);
    float* H = reinterpret_cast<float*>(base + 2 * np + nk);
    NMF_CUDA_TRY(p, cudaMemcpyAsync(X, Xh, sizeof(float) * (size_t)p->N * p->P, cudaMemcpyHostToDevice, p->stream));
    NMF_CUDA_TRY(p, cudaMemcpyAsync(Om, Oh, sizeof(float) * (size_t)p->N * p->P, cudaMemcpyHostToDevice, p->stream));
    NMF_CUDA_TRY(p, cudaMemcpyAsync(W, Wh, sizeof(float) * (size_t)p->N * p->K, cudaMemcpyHostToDevice, p->stream));
    NMF_CUDA_TRY(p, cudaMemcpyAsync(H, Hh, sizeof(float) * (size_t)p->K * p->P, cudaMemcpyHostToDevice, p->stream));
    rc = fit_common(p, X, Om, W, H, iters, 1);
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaMemcpyAsync(Wh, W, sizeof(float) * (size_t)p->N * p->K, cudaMemcpyDeviceToHost, p->stream));
    NMF_CUDA_TRY(p, cudaMemcpyAsync(Hh, H, sizeof(float) * (size_t)p->K * p->P, cudaMemcpyDeviceToHost, p->stream));
    NMF_CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    return NMF_OK;
}

int nmf_project_subtract_host(nmf_plan* p, const float* H, const float* Th, const float* oh,
                              float* Ch, float fill, float* outh, int M, int iters) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!H || !Th || !Ch || !outh || M < 1 || M > p->max_targets || iters < 0) return NMF_ERR_INVALID_ARG;
    if (int rcd = check_device(p)) return rcd;
    const size_t mp = nmf_align_up(sizeof(float) * (size_t)M * p->P, 256);
    const size_t mk = nmf_align_up(sizeof(float) * (size_t)M * p->K, 256);
    int rc = ensure_stage(p, 3 * mp + mk);
    if (rc) return rc;
    rc = ensure_own_ws(p);
    if (rc) return rc;
    char* base = static_cast<char*>(p->stage);
    float* T = reinterpret_cast<float*>(base);
    float* om = oh ? reinterpret_cast<float*>(base + mp) : nullptr;
    float* out = reinterpret_cast<float*>(base + 2 * mp);
    float* C = reinterpret_cast<float*>(base + 3 * mp);
    NMF_CUDA_TRY(p, cudaMemcpyAsync(T, Th, sizeof(float) * (size_t)M * p->P, cudaMemcpyHostToDevice, p->stream));
    if (oh) NMF_CUDA_TRY(p, cudaMemcpyAsync(om, oh, sizeof(float) * (size_t)M * p->P, cudaMemcpyHostToDevice, p->stream));
    NMF_CUDA_TRY(p, cudaMemcpyAsync(C, Ch, sizeof(float) * (size_t)M * p->K, cudaMemcpyHostToDevice, p->stream));
    rc = nmf_project(p, H, T, om, C, M, iters);
    if (rc) return rc;
    rc = nmf_subtract(p, H, T, C, om, nullptr, fill, out, M);
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaMemcpyAsync(Ch, C, sizeof(float) * (size_t)M * p->K, cudaMemcpyDeviceToHost, p->stream));
    NMF_CUDA_TRY(p, cudaMemcpyAsync(outh, out, sizeof(float) * (size_t)M * p->P, cudaMemcpyDeviceToHost, p->stream));
    NMF_CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    return NMF_OK;
}

int nmf_ref_distance(nmf_plan* p, const float* T, const float* ot, const float* X, const float* Om, int M,
                     float* dist) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!T || !X || !dist || M < 1) return NMF_ERR_INVALID_ARG;
    if (misaligned(T) || misaligned(X) || misaligned(dist) || (ot && misaligned(ot)) || (Om && misaligned(Om)))
        return NMF_ERR_ALIGNMENT;
    int rc = check_ws(p);
    if (rc) return rc;
    return nmf_select_distance(p, T, ot, X, Om, M, dist);
}

int nmf_ref_select(nmf_plan* p, const float* dist, int M, int n_sel, int* idx) {
    if (!p) return NMF_ERR_INVALID_ARG;
    if (p->sticky) return p->sticky;
    if (!dist || !idx || M < 1 || n_sel < 1 || n_sel > p->N) return NMF_ERR_INVALID_ARG;
    int rc = check_device(p);
    if (rc) return rc;
    return nmf_select_topn(p, dist, M, n_sel, idx);
}

long long nmf_plan_launch_count(const nmf_plan* p) { return p ? p->launches : 0; }

const char* nmf_status_string(int code) {
    switch (code) {
        case NMF_OK: return "NMF_OK";
        case NMF_ERR_INVALID_ARG: return "NMF_ERR_INVALID_ARG: null pointer or size out of range";
        case NMF_ERR_ALIGNMENT: return "NMF_ERR_ALIGNMENT: pointer not 16-byte aligned or P % 4 != 0";
        case NMF_ERR_UNSUPPORTED: return "NMF_ERR_UNSUPPORTED: shape beyond the compiled limits";
        case NMF_ERR_WORKSPACE: return "NMF_ERR_WORKSPACE: workspace missing or too small";
        case NMF_ERR_ARCH: return "NMF_ERR_ARCH: device is not compute capability 10.x (B200)";
        case NMF_ERR_CUDA: return "NMF_ERR_CUDA: CUDA runtime or launch error";
        case NMF_ERR_STATIC_LIMIT: return "NMF_ERR_STATIC_LIMIT: P beyond the fixed scratch of nmf_objective_static (NMF_STATIC_MAX_P = 2048^2 pixels)";
        default: return "unknown nmf status";
    }
}

const char* nmf_plan_last_cuda_error(const nmf_plan* p) { return p ? p->cuda_msg.c_str() : ""; }

}  // extern "C"

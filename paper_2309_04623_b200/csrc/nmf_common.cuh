// nmf_common.cuh -- shared host/device declarations of the sm_100a NMF library.
// (Library-internal; the public boundary is include/nmf.h.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include "../../include/nmf.h"

#define NMF_MAX_DEVICES 64   // plan->device is checked against this at plan creation
#define NMF_EPS 1e-30f   // ratio guard: num / max(den, NMF_EPS)   (reading G4)

// ---------------------------------------------------------------------------
// plan
// ---------------------------------------------------------------------------
struct nmf_plan {
    int N = 0, K = 0, batch = 1, max_targets = 0;
    long long P = 0;
    int device = 0;
    int num_sms = 148;
    cudaStream_t stream = nullptr;
    void* ws = nullptr;
    size_t ws_bytes = 0;
    size_t ws_needed = 0;
    int variant_req = 0;          // 0 auto, 1 generic, 2 fused FFMA, 3 fused tensor core, 4 split tensor core, 5 streaming FP32, 6 resident
    long long launches = 0;
    int sticky = 0;               // first CUDA error seen (nmf_status)
    std::string cuda_msg;

    // generic-path geometry (see nmf_generic.cu)
    int g_kc = 0, g_ks = 0;       // per-thread K chunk, lanes per item
    int g_parts_fit = 0;          // pixel-range partitions of the W half-step (fit)
    int g_parts_proj = 0;         // same for projection
    // fused-path geometry (see nmf_fused.cu)
    int f_kp = 0;                 // padded K of the fused instantiation (0 = unavailable)
    int f_ctas = 0;               // persistent CTAs per problem
    int f_threads = 0;            // CTA size = pixels per tile
    int f_fpw = 0;                // frames per warp in the W half
    // tensor-core path geometry (see nmf_tcfit.cu)
    int t_ctas = 0;               // persistent CTAs per problem (0 = unavailable)
    // split tensor-core path (see nmf_tcsplit.cu)
    bool s_ok = false;
    // streaming FP32 kernel for K <= 8 (see nmf_stream.cu)
    bool st_ok = false;
    // all iterations in one cooperative launch, problem resident on chip (see nmf_resident.cu)
    bool rs_ok = false;
    // host staging for the *_host entry points (plan-owned device buffers)
    void* stage = nullptr;
    size_t stage_bytes = 0;
    bool stage_user = false;      // the staging buffer was handed over by the caller (nmf_plan_set_staging)
    void* own_ws = nullptr;       // workspace allocated by a *_host call when none was set
    double* host_scratch = nullptr;   // 8 pinned doubles: results read back by nmf_objective / nmf_fit_tol
    // iteration loop as a CUDA graph (nmf_run_iterations): one instantiated graph of `g_unroll` iterations, kept
    // while the same call (kernel family, buffers, shape) is repeated
    cudaStream_t cap_stream = nullptr;    // plan-owned stream the graph is captured on (the legacy default stream cannot be)
    cudaGraphExec_t g_exec = nullptr;
    const void* g_key[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int g_rows = 0, g_batch = 0, g_unroll = 0, g_kind = 0;
    long long g_launches = 0;             // kernel launches of one replay
};

static inline int nmf_cuda_fail(nmf_plan* p, cudaError_t e) {
    if (p && !p->sticky) { p->sticky = NMF_ERR_CUDA; p->cuda_msg = cudaGetErrorString(e); }
    return NMF_ERR_CUDA;
}
#define NMF_CUDA_TRY(plan, expr)                                   \
    do { cudaError_t _e = (expr);                                  \
         if (_e != cudaSuccess) return nmf_cuda_fail((plan), _e); } while (0)

static inline size_t nmf_align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---------------------------------------------------------------------------
// iteration loop without per-launch host work
// ---------------------------------------------------------------------------
// Runs `iters` repetitions of `one()` -- which enqueues ONE iteration's kernels on plan->stream and returns an NMF
// status -- in stream order on plan->stream.  From NMF_GRAPH_MIN iterations up, min(iters, NMF_GRAPH_UNROLL)
// repetitions are captured once into a CUDA graph (on a plan-owned capture stream), instantiated, and replayed
// iters / unroll times; the remainder is enqueued directly.  The instantiated graph is kept in the plan and reused
// while the same call (kind, buffers, rows, batch) comes again.  Inside someone else's capture the plain loop runs.
#define NMF_GRAPH_MIN 8
#define NMF_GRAPH_UNROLL 50
template <class F>
static inline int nmf_run_iterations(nmf_plan* p, int kind, const void* k0, const void* k1, const void* k2, const void* k3,
                                     const void* k4, int rows, int batch, int iters, F one) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const bool capturing = cudaStreamIsCapturing(p->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone;
    if (capturing) (void)cudaGetLastError();
    int done = 0;
    if (!capturing && iters >= NMF_GRAPH_MIN) {
        const int unroll = iters < NMF_GRAPH_UNROLL ? iters : NMF_GRAPH_UNROLL;
        const void* key[6] = {k0, k1, k2, k3, k4, reinterpret_cast<const void*>(p->ws)};
        bool hit = p->g_exec && p->g_kind == kind && p->g_rows == rows && p->g_batch == batch && p->g_unroll == unroll;
        for (int i = 0; i < 6 && hit; ++i) hit = p->g_key[i] == key[i];
        if (!hit) {
            if (p->g_exec) { cudaGraphExecDestroy(p->g_exec); p->g_exec = nullptr; }
            if (!p->cap_stream) NMF_CUDA_TRY(p, cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
            cudaStream_t user = p->stream;
            const long long l0 = p->launches;
            NMF_CUDA_TRY(p, cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal));
            p->stream = p->cap_stream;
            int rc = NMF_OK;
            for (int u = 0; u < unroll && rc == NMF_OK; ++u) rc = one();
            p->stream = user;
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamEndCapture(p->cap_stream, &graph);
            p->g_launches = p->launches - l0;
            p->launches = l0;
            if (rc != NMF_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
            NMF_CUDA_TRY(p, e);
            e = cudaGraphInstantiate(&p->g_exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { p->g_exec = nullptr; return nmf_cuda_fail(p, e); }
            for (int i = 0; i < 6; ++i) p->g_key[i] = key[i];
            p->g_kind = kind; p->g_rows = rows; p->g_batch = batch; p->g_unroll = unroll;
        }
        for (; done + p->g_unroll <= iters; done += p->g_unroll) {
            NMF_CUDA_TRY(p, cudaGraphLaunch(p->g_exec, p->stream));
            p->launches += p->g_launches;
        }
    }
    for (; done < iters; ++done) {
        int rc = one();
        if (rc) return rc;
    }
    return NMF_OK;
}

// ---------------------------------------------------------------------------
// launchers implemented in the .cu files (all enqueue on plan->stream)
// ---------------------------------------------------------------------------
// generic two-kernel path
void   nmf_generic_configure(nmf_plan* p);
size_t nmf_generic_workspace(const nmf_plan* p);
int    nmf_generic_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H,
                       int iters, int batch);
int    nmf_generic_project(nmf_plan* p, const float* H, const float* T, const float* om,
                           float* C, int M, int iters);
// fixed-order fp64 reduction of `parts` partial slabs [batch][parts][2][rows][KT] + W update
int    nmf_launch_w_update(nmf_plan* p, const float* slab, float* W, int rows, int K, int KT,
                           int parts, int batch);
// fused per-pixel-tile path
void   nmf_fused_configure(nmf_plan* p);
size_t nmf_fused_workspace(const nmf_plan* p);
bool   nmf_fused_available(const nmf_plan* p);
int    nmf_fused_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H,
                     int iters, int batch);
// tcgen05 tensor-core fused path (BF16x3 split, FP32 accumulation in TMEM)
void   nmf_tc_configure(nmf_plan* p);
size_t nmf_tc_workspace(const nmf_plan* p);
bool   nmf_tc_available(const nmf_plan* p);
int    nmf_tc_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H,
                  int iters, int batch);
int    nmf_tc_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C,
                      int M, int iters);
// split tensor-core path: H half-step kernel + W half-step kernel, K <= 128 (nmf_tcsplit.cu)
void   nmf_tcsplit_configure(nmf_plan* p);
size_t nmf_tcsplit_workspace(const nmf_plan* p);
bool   nmf_tcsplit_available(const nmf_plan* p);
int    nmf_tcsplit_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H,
                       int iters, int batch);
int    nmf_tcsplit_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C,
                           int M, int iters);
// streaming FP32 kernel, one launch per iteration, K <= 8 (nmf_stream.cu)
void   nmf_stream_configure(nmf_plan* p);
size_t nmf_stream_workspace(const nmf_plan* p);
bool   nmf_stream_available(const nmf_plan* p);
int    nmf_stream_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H,
                      int iters, int batch);
// whole fit in one cooperative launch for problems that stay on chip: K <= 8, N <= 64, P <= 128 x SMs (nmf_resident.cu)
void   nmf_resident_configure(nmf_plan* p);
size_t nmf_resident_workspace(const nmf_plan* p);
bool   nmf_resident_available(const nmf_plan* p);
int    nmf_resident_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters);
// closest-frame reference selection (nmf_select.cu)
size_t nmf_select_workspace(const nmf_plan* p);
int    nmf_select_distance(nmf_plan* p, const float* T, const float* ot, const float* X, const float* Om,
                           int M, float* D);
int    nmf_select_topn(nmf_plan* p, const float* D, int M, int n_sel, int* idx);
// auxiliaries
size_t nmf_aux_workspace(const nmf_plan* p);
int    nmf_aux_subtract(nmf_plan* p, const float* H, const float* T, const float* C,
                        const float* om, const float* factor, float fill, float* out, int M);
int    nmf_aux_objective(nmf_plan* p, const float* X, const float* Om, const float* W,
                         const float* H, double* out_host);
int    nmf_aux_objective_dev(nmf_plan* p, const float* X, const float* Om, const float* W,
                             const float* H, double* f_dev);
int    nmf_aux_fit_tol(nmf_plan* p, int (*fit)(nmf_plan*, const float*, const float*, float*, float*, int),
                       const float* X, const float* Om, float* W, float* H, int max_iters, int check_every,
                       double tol, int* iters_done, double* f_last);
int    nmf_aux_derotate_stack(nmf_plan* p, const float* R, const float* om, const float* angle, int ny, int nx,
                              float fill, float* out, int* count, int M);

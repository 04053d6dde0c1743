// nmf_aux.cu -- PSF subtraction, the objective of Eq. 2 reduced on the device
// in fp64 in a fixed order, the tolerance test of the stopping rule (8(f) NEXT-3) and
// derotation + stacking of the residual frames (8(f) NEXT-4).
#include "nmf_common.cuh"

namespace {

constexpr int SUB_MC = 32;      // science frames per pass (accumulators per thread)
constexpr int SUB_THREADS = 128;
constexpr int SUB_MH = 8;       // frames per CTA (accumulator rows per thread)
constexpr int SUB_PX = 4;       // pixels per thread (one 128-bit column segment of H, T, omega, out)
constexpr int OBJ_THREADS = 128;

// out[m,p] = t[m,p] - f[m] * sum_k c[m,k] H[k,p]; `fill` where omega[m,p] == 0.
// Four pixels per thread (128-bit loads of H, T, omega; 128-bit stores), SUB_MC frames per launch handled as
// SUB_MC / SUB_MH groups of SUB_MH = 8 frames: 32 accumulators, 63 registers, eight CTAs per SM overlap one another's
// compute (K loop) and streaming (T, omega, out) phases (16 frames per CTA: 0.169 ms, 8: 0.159 ms, 4: 0.37 ms -- the
// coefficient loads and the 8-fold L2 read of H then dominate).  The frame groups of a pixel segment
// are taken by ADJACENT CTAs (blockIdx.x = segment * groups + group): they run at the same time, so the H columns the
// later ones read are in L2 (as two passes of one CTA they were 74 MB of other CTAs' traffic apart and missed: 1.3x
// the algorithmic DRAM bytes).  Coefficients are 128-bit shared-memory broadcasts (cs[k][m]).
__global__ void __launch_bounds__(SUB_THREADS, 8)
k_subtract(const float* __restrict__ H, const float* __restrict__ T, const float* __restrict__ C,
           const float* __restrict__ om, const float* __restrict__ factor, float fill,
           float* __restrict__ out, int M, long long P, int K, int m0) {
    extern __shared__ __align__(16) float cs[];   // [K][SUB_MC]
    const int mc = min(SUB_MC, M - m0);
    for (int i = threadIdx.x; i < SUB_MC * K; i += SUB_THREADS) {
        const int k = i / SUB_MC, m = i - k * SUB_MC;
        cs[i] = m < mc ? C[(size_t)(m0 + m) * K + k] : 0.f;
    }
    __syncthreads();
    constexpr int NGRP = SUB_MC / SUB_MH;
    const long long p = ((long long)(blockIdx.x / NGRP) * SUB_THREADS + threadIdx.x) * SUB_PX;
    if (p >= P) return;                            // P % 4 == 0: a segment is all in or all out
    const int mh = (int)(blockIdx.x % NGRP) * SUB_MH;
    if (mh < mc) {
        float acc[SUB_MH][SUB_PX];
#pragma unroll
        for (int m = 0; m < SUB_MH; ++m)
#pragma unroll
            for (int q = 0; q < SUB_PX; ++q) acc[m][q] = 0.f;
        const float* hp = H + p;
        constexpr int KU = 5;                      // H rows in flight per thread (10: spills or fewer CTAs per SM, slower)
        for (int k0 = 0; k0 < K; k0 += KU) {
            float4 hv[KU];
#pragma unroll
            for (int u = 0; u < KU; ++u)
                hv[u] = (k0 + u < K) ? __ldg(reinterpret_cast<const float4*>(hp + (size_t)(k0 + u) * P)) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int u = 0; u < KU; ++u) {
                if (k0 + u < K) {
                    const float4 h = hv[u];
                    const float* ck = cs + (k0 + u) * SUB_MC + mh;
#pragma unroll
                    for (int m4 = 0; m4 < SUB_MH / 4; ++m4) {
                        const float4 c = *reinterpret_cast<const float4*>(ck + 4 * m4);
                        const float cc[4] = {c.x, c.y, c.z, c.w};
#pragma unroll
                        for (int v = 0; v < 4; ++v) {
                            acc[4 * m4 + v][0] = fmaf(cc[v], h.x, acc[4 * m4 + v][0]);
                            acc[4 * m4 + v][1] = fmaf(cc[v], h.y, acc[4 * m4 + v][1]);
                            acc[4 * m4 + v][2] = fmaf(cc[v], h.z, acc[4 * m4 + v][2]);
                            acc[4 * m4 + v][3] = fmaf(cc[v], h.w, acc[4 * m4 + v][3]);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int m = 0; m < SUB_MH; ++m) {
            if (mh + m < mc) {
                const size_t i = (size_t)(m0 + mh + m) * P + p;
                const float f = factor ? factor[m0 + mh + m] : 1.f;
                const float4 t = __ldg(reinterpret_cast<const float4*>(T + i));
                float4 o = make_float4(1.f, 1.f, 1.f, 1.f);
                if (om) o = __ldg(reinterpret_cast<const float4*>(om + i));
                float4 r;                          // omega == 0: T may hold NaN/Inf there (G5) -> select
                r.x = o.x > 0.f ? t.x - f * acc[m][0] : fill;
                r.y = o.y > 0.f ? t.y - f * acc[m][1] : fill;
                r.z = o.z > 0.f ? t.z - f * acc[m][2] : fill;
                r.w = o.w > 0.f ? t.w - f * acc[m][3] : fill;
                *reinterpret_cast<float4*>(out + i) = r;
            }
        }
    }
}

// sum_{Om>0} Om (X - W H)^2 in fp64; one pixel per thread, per-block partial.
__global__ void __launch_bounds__(OBJ_THREADS)
k_objective(const float* __restrict__ X, const float* __restrict__ Om, const float* __restrict__ W,
            const float* __restrict__ H, double* __restrict__ partial, int N, long long P, int K) {
    extern __shared__ __align__(16) float smem[];
    float* ws = smem;                       // [N][K]
    float* hs = smem + (size_t)N * K;       // [K][OBJ_THREADS]
    __shared__ double red[OBJ_THREADS / 32];
    for (int i = threadIdx.x; i < N * K; i += OBJ_THREADS) ws[i] = W[i];
    const long long p = (long long)blockIdx.x * OBJ_THREADS + threadIdx.x;
    const bool active = p < P;
    for (int k = 0; k < K; ++k) hs[k * OBJ_THREADS + threadIdx.x] = active ? H[(size_t)k * P + p] : 0.f;
    __syncthreads();
    double f = 0.0;
    if (active) {
        for (int n = 0; n < N; ++n) {
            const float o = Om[(size_t)n * P + p];
            if (!(o > 0.f)) continue;
            double s = 0.0;
            for (int k = 0; k < K; ++k) s += (double)ws[n * K + k] * (double)hs[k * OBJ_THREADS + threadIdx.x];
            const double d = (double)X[(size_t)n * P + p] - s;
            f += (double)o * d * d;
        }
    }
    for (int d = 16; d > 0; d >>= 1) f += __shfl_xor_sync(0xffffffffu, f, d);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = f;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < OBJ_THREADS / 32; ++w) t += red[w];
        partial[blockIdx.x] = t;
    }
}

// fixed-order sum of the per-block partials: thread i adds partials i, i + 256, ... in order, thread 0 then adds the
// 256 thread sums in order (bitwise reproducible); one block
constexpr int RED_THREADS = 256;
__global__ void __launch_bounds__(RED_THREADS)
k_objective_reduce(const double* __restrict__ partial, int n, double* __restrict__ f_out) {
    __shared__ double sh[RED_THREADS];
    double a = 0.0;
    for (int i = threadIdx.x; i < n; i += RED_THREADS) a += partial[i];
    sh[threadIdx.x] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < RED_THREADS; ++i) t += sh[i];
        *f_out = t;
    }
}

// stopping test of reading G21: stop = |f_prev - f_cur| < tol * f_prev; then f_prev <- f_cur.
// res[0] = f_prev (in/out), res[1] = f_cur (in), res[2] = stop flag as a double (out)
__global__ void k_tol_check(double* res, double tol) {
    const double fp = res[0], fc = res[1];
    res[2] = (fabs(fp - fc) < tol * fp) ? 1.0 : 0.0;
    res[0] = fc;
}

// sine / cosine of an angle in degrees, exact at multiples of 90 degrees (reading G22): fold to the nearest multiple
// of 90, evaluate the remainder |r| <= 45 degrees in fp64, rotate by the quadrant
__device__ __forceinline__ void sincos_deg(double deg, double* s, double* c) {
    double a = fmod(deg, 360.0);
    if (a < 0.0) a += 360.0;
    const int k = (int)floor(a / 90.0 + 0.5);
    const double r = (a - 90.0 * k) * (3.14159265358979323846 / 180.0);
    double sr, cr;
    sincos(r, &sr, &cr);
    switch (k & 3) {
        case 0: *s = sr;  *c = cr;  break;
        case 1: *s = cr;  *c = -sr; break;
        case 2: *s = -sr; *c = -cr; break;
        default: *s = -cr; *c = sr; break;
    }
}

// derotate + stack (readings G22-G24): one output pixel per thread, 32 x 8 pixel tile per CTA; frame m rotated by
// angle[m] about the pixel (ny / 2, nx / 2), bilinear over the neighbours with weight > 1e-6, a sample counts only if
// all of those are inside the image and have omega > 0; out = mean over the frames with a sample, else `fill`.
// Source coordinates and weights in fp64 (they decide which pixels are read), the weighted sum in fp32.
constexpr int ROT_TX = 32, ROT_TY = 8, ROT_MC = 128;
__global__ void __launch_bounds__(ROT_TX * ROT_TY)
k_derotate_stack(const float* __restrict__ R, const float* __restrict__ om, const float* __restrict__ angle,
                 int M, int ny, int nx, float fill, float* __restrict__ out, int* __restrict__ count) {
    __shared__ double sn[ROT_MC], cs[ROT_MC];
    const int tid = threadIdx.y * ROT_TX + threadIdx.x;
    const int x = blockIdx.x * ROT_TX + threadIdx.x, y = blockIdx.y * ROT_TY + threadIdx.y;
    const bool in = x < nx && y < ny;
    const size_t P = (size_t)ny * nx;
    const int cy = ny / 2, cx = nx / 2;
    const double dx = x - cx, dy = y - cy;
    float sum = 0.f;
    int cnt = 0;
    for (int m0 = 0; m0 < M; m0 += ROT_MC) {
        const int mc = min(ROT_MC, M - m0);
        __syncthreads();
        if (tid < mc) sincos_deg((double)angle[m0 + tid], &sn[tid], &cs[tid]);
        __syncthreads();
        if (!in) continue;
        for (int m = 0; m < mc; ++m) {
            const double xs = cx + cs[m] * dx + sn[m] * dy;
            const double ys = cy - sn[m] * dx + cs[m] * dy;
            const double x0 = floor(xs), y0 = floor(ys);
            const double fx = xs - x0, fy = ys - y0;
            const double w[4] = {(1.0 - fx) * (1.0 - fy), fx * (1.0 - fy), (1.0 - fx) * fy, fx * fy};
            const float* Rm = R + (size_t)(m0 + m) * P;
            const float* om_m = om ? om + (size_t)(m0 + m) * P : nullptr;
            bool valid = true;
            float v = 0.f;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (!(w[i] > 1e-6)) continue;
                const double xi = x0 + (i & 1), yi = y0 + (i >> 1);
                if (xi < 0 || xi >= nx || yi < 0 || yi >= ny) { valid = false; continue; }
                const size_t j = (size_t)yi * nx + (size_t)xi;
                if (om_m && !(__ldg(om_m + j) > 0.f)) { valid = false; continue; }
                if (valid) v = fmaf((float)w[i], __ldg(Rm + j), v);     // (a masked pixel's value is never read)
            }
            if (valid) { sum += v; ++cnt; }
        }
    }
    if (in) {
        out[(size_t)y * nx + x] = cnt ? sum / (float)cnt : fill;
        if (count) count[(size_t)y * nx + x] = cnt;
    }
}

}  // namespace

size_t nmf_aux_workspace(const nmf_plan* p) {
    // objective partials (one double per block) + 4 doubles: f_prev, f_cur, stop flag, spare
    return sizeof(double) * ((size_t)((p->P + OBJ_THREADS - 1) / OBJ_THREADS) + 4);
}

int nmf_aux_subtract(nmf_plan* p, const float* H, const float* T, const float* C, const float* om,
                     const float* factor, float fill, float* out, int M) {
    const long long per_cta = (long long)SUB_THREADS * SUB_PX;
    const unsigned grid = (unsigned)((p->P + per_cta - 1) / per_cta) * (SUB_MC / SUB_MH);
    const size_t smem = sizeof(float) * SUB_MC * p->K;
    for (int m0 = 0; m0 < M; m0 += SUB_MC) {
        k_subtract<<<grid, SUB_THREADS, smem, p->stream>>>(H, T, C, om, factor, fill, out, M, p->P, p->K, m0);
        p->launches++;
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

// scratch doubles at the very end of the workspace: [0] f_prev, [1] f_cur, [2] stop flag
static double* aux_scratch(nmf_plan* p) {
    return reinterpret_cast<double*>(static_cast<char*>(p->ws) + p->ws_needed) - 4;
}

// the cost of Eq. 2 at (W, H) into device memory `f_dev` (fp64, fixed-order: bitwise reproducible); asynchronous
int nmf_aux_objective_dev(nmf_plan* p, const float* X, const float* Om, const float* W, const float* H, double* f_dev) {
    const unsigned grid = (unsigned)((p->P + OBJ_THREADS - 1) / OBJ_THREADS);
    const size_t smem = sizeof(float) * ((size_t)p->N * p->K + (size_t)p->K * OBJ_THREADS);
    static bool attr_done[NMF_MAX_DEVICES] = {};   // function attributes are per device
    if (!attr_done[p->device]) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_objective, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_done[p->device] = true;
    }
    // objective partials live at the tail of the workspace
    double* partial = reinterpret_cast<double*>(static_cast<char*>(p->ws) + (p->ws_needed - nmf_aux_workspace(p)));
    k_objective<<<grid, OBJ_THREADS, smem, p->stream>>>(X, Om, W, H, partial, p->N, p->P, p->K);
    k_objective_reduce<<<1, RED_THREADS, 0, p->stream>>>(partial, (int)grid, f_dev);
    p->launches += 2;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

int nmf_aux_objective(nmf_plan* p, const float* X, const float* Om, const float* W, const float* H,
                      double* out_host) {
    double* sc = aux_scratch(p);
    int rc = nmf_aux_objective_dev(p, X, Om, W, H, sc + 1);
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaMemcpyAsync(p->host_scratch, sc + 1, sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    NMF_CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    *out_host = p->host_scratch[0];
    return NMF_OK;
}

// fit with the tolerance stop of reading G21: blocks of `check_every` iterations, each followed by the device-side
// cost + stopping test; the host reads the 3-double result once per block (not per iteration)
int nmf_aux_fit_tol(nmf_plan* p, int (*fit)(nmf_plan*, const float*, const float*, float*, float*, int),
                    const float* X, const float* Om, float* W, float* H, int max_iters, int check_every, double tol,
                    int* iters_done, double* f_last) {
    double* sc = aux_scratch(p);
    int rc = nmf_aux_objective_dev(p, X, Om, W, H, sc);            // f_prev = f_0
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaMemcpyAsync(p->host_scratch, sc, sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    int it = 0;
    bool checked = false;
    while (it < max_iters) {
        const int n = (max_iters - it < check_every) ? max_iters - it : check_every;
        rc = fit(p, X, Om, W, H, n);
        if (rc) return rc;
        it += n;
        if (n < check_every) break;                                // max_iters reached between two checks
        rc = nmf_aux_objective_dev(p, X, Om, W, H, sc + 1);
        if (rc) return rc;
        k_tol_check<<<1, 1, 0, p->stream>>>(sc, tol);
        p->launches++;
        NMF_CUDA_TRY(p, cudaMemcpyAsync(p->host_scratch, sc, 3 * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
        NMF_CUDA_TRY(p, cudaStreamSynchronize(p->stream));
        checked = true;
        if (p->host_scratch[2] != 0.0) break;
    }
    if (!checked) NMF_CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    *iters_done = it;
    if (f_last) *f_last = p->host_scratch[0];
    return NMF_OK;
}

int nmf_aux_derotate_stack(nmf_plan* p, const float* R, const float* om, const float* angle, int ny, int nx, float fill,
                           float* out, int* count, int M) {
    dim3 grid((nx + ROT_TX - 1) / ROT_TX, (ny + ROT_TY - 1) / ROT_TY), block(ROT_TX, ROT_TY);
    k_derotate_stack<<<grid, block, 0, p->stream>>>(R, om, angle, M, ny, nx, fill, out, count);
    p->launches++;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

// =====================================================================================================================
// nmf_objective_static: the cost of Eq. 2 WITHOUT a plan, a workspace or any allocation (include/nmf.h).
// The per-block partial sums of k_objective live in a file-scope device array of fixed size; every device that loads
// the library holds it (256 KB) until the process exits.
// =====================================================================================================================
namespace {

constexpr long long STATIC_MAX_BLOCKS = (NMF_STATIC_MAX_P + OBJ_THREADS - 1) / OBJ_THREADS;   // 32768 doubles = 256 KB
constexpr size_t STATIC_MAX_SMEM = 200 * 1024;                                                 // as nmf_aux_objective_dev

static __device__ __align__(256) double g_static_partial[STATIC_MAX_BLOCKS];

// In host code `g_static_partial` is a host-side stand-in for the symbol, not a device address: the address the
// kernels need comes from cudaGetSymbolAddress, once per device, with that device current.
struct StaticDev { bool ready = false; double* partial = nullptr; };
StaticDev g_static_dev[NMF_MAX_DEVICES];

int static_setup(int device, double** partial) {
    StaticDev& d = g_static_dev[device];
    if (!d.ready) {                                       // (plain flag: the calls below are idempotent, a race repeats them)
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess) return NMF_ERR_CUDA;
        if (major != 10) return NMF_ERR_ARCH;
        double* ptr = nullptr;
        if (cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_static_partial) != cudaSuccess || !ptr) return NMF_ERR_CUDA;
        if (cudaFuncSetAttribute(k_objective, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)STATIC_MAX_SMEM) != cudaSuccess)
            return NMF_ERR_CUDA;
        d.partial = ptr;
        d.ready = true;
    }
    *partial = d.partial;
    return NMF_OK;
}

}  // namespace

extern "C" int nmf_objective_static(const float* X, const float* Omega, const float* W, const float* H, int N, long long P,
                                    int K, double* f_out_dev, void* stream) {
    if (!X || !Omega || !W || !H || !f_out_dev || N < 1 || P < 1 || K < 1) return NMF_ERR_INVALID_ARG;
    if (N > NMF_MAX_N || K > NMF_MAX_K) return NMF_ERR_UNSUPPORTED;
    const size_t smem = sizeof(float) * ((size_t)N * K + (size_t)K * OBJ_THREADS);
    if (P > NMF_STATIC_MAX_P || smem > STATIC_MAX_SMEM) return NMF_ERR_STATIC_LIMIT;
    int device = 0;
    if (cudaGetDevice(&device) != cudaSuccess) return NMF_ERR_CUDA;
    if (device < 0 || device >= NMF_MAX_DEVICES) return NMF_ERR_UNSUPPORTED;
    double* partial = nullptr;
    const int rc = static_setup(device, &partial);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)((P + OBJ_THREADS - 1) / OBJ_THREADS);
    // every partial that is read (blocks 0 .. grid - 1) is written by this call's first kernel: nothing left over from
    // an earlier call is read, so nothing needs clearing
    k_objective<<<grid, OBJ_THREADS, smem, st>>>(X, Omega, W, H, partial, N, P, K);
    k_objective_reduce<<<1, RED_THREADS, 0, st>>>(partial, (int)grid, f_out_dev);
    return cudaGetLastError() == cudaSuccess ? NMF_OK : NMF_ERR_CUDA;
}

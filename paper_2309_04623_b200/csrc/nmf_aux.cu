// nmf_aux.cu -- PSF subtraction and the diagnostic
// objective of Eq. 2.
#include "nmf_common.cuh"

namespace {

constexpr int SUB_MC = 32;      // science frames per pass (accumulators per thread)
constexpr int SUB_THREADS = 128;
constexpr int SUB_MH = 16;      // frames per register pass
constexpr int SUB_PX = 4;       // pixels per thread (one 128-bit column segment of H, T, omega, out)
constexpr int OBJ_THREADS = 128;

// out[m,p] = t[m,p] - f[m] * sum_k c[m,k] H[k,p]; `fill` where omega[m,p] == 0.
// Four pixels per thread (128-bit loads of H, T, omega; 128-bit stores), SUB_MC frames per launch handled as
// SUB_MC / SUB_MH passes of SUB_MH frames: 64 accumulators keep the register count near 100, so five CTAs per SM
// overlap one another's compute (K loop) and streaming (T, omega, out) phases; the H columns of the second pass
// come back from L1 / L2.  Coefficients are 128-bit shared-memory broadcasts (cs[k][m]).
__global__ void __launch_bounds__(SUB_THREADS, 5)
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
    const long long p = ((long long)blockIdx.x * SUB_THREADS + threadIdx.x) * SUB_PX;
    if (p >= P) return;                            // P % 4 == 0: a segment is all in or all out
    for (int mh = 0; mh < mc; mh += SUB_MH) {
        float acc[SUB_MH][SUB_PX];
#pragma unroll
        for (int m = 0; m < SUB_MH; ++m)
#pragma unroll
            for (int q = 0; q < SUB_PX; ++q) acc[m][q] = 0.f;
        const float* hp = H + p;
        constexpr int KU = 5;                      // H rows in flight per thread
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

}  // namespace

size_t nmf_aux_workspace(const nmf_plan* p) {
    return sizeof(double) * (size_t)((p->P + OBJ_THREADS - 1) / OBJ_THREADS);
}

int nmf_aux_subtract(nmf_plan* p, const float* H, const float* T, const float* C, const float* om,
                     const float* factor, float fill, float* out, int M) {
    const long long per_cta = (long long)SUB_THREADS * SUB_PX;
    const unsigned grid = (unsigned)((p->P + per_cta - 1) / per_cta);
    const size_t smem = sizeof(float) * SUB_MC * p->K;
    for (int m0 = 0; m0 < M; m0 += SUB_MC) {
        k_subtract<<<grid, SUB_THREADS, smem, p->stream>>>(H, T, C, om, factor, fill, out, M, p->P, p->K, m0);
        p->launches++;
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

int nmf_aux_objective(nmf_plan* p, const float* X, const float* Om, const float* W, const float* H,
                      double* out_host) {
    const unsigned grid = (unsigned)((p->P + OBJ_THREADS - 1) / OBJ_THREADS);
    const size_t smem = sizeof(float) * ((size_t)p->N * p->K + (size_t)p->K * OBJ_THREADS);
    bool attr_done = false;   // function attributes are per device: set on every call (cheap)
    if (!attr_done) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_objective, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_done = true;
    }
    // objective partials live at the tail of the workspace
    double* partial = reinterpret_cast<double*>(static_cast<char*>(p->ws) + (p->ws_needed - nmf_aux_workspace(p)));
    k_objective<<<grid, OBJ_THREADS, smem, p->stream>>>(X, Om, W, H, partial, p->N, p->P, p->K);
    p->launches++;
    NMF_CUDA_TRY(p, cudaGetLastError());
    double* host = nullptr;
    NMF_CUDA_TRY(p, cudaMallocHost(&host, sizeof(double) * grid));
    cudaError_t e = cudaMemcpyAsync(host, partial, sizeof(double) * grid, cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) { cudaFreeHost(host); return nmf_cuda_fail(p, e); }
    double f = 0.0;
    for (unsigned i = 0; i < grid; ++i) f += host[i];   // fixed order
    cudaFreeHost(host);
    *out_host = f;
    return NMF_OK;
}

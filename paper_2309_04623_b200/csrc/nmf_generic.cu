// nmf_generic.cu -- generic two-kernel path for any N <= 256, K <= 128.
//
// One iteration = H half-step kernel, W half-step partial kernel, fixed-order
// reduction + W update kernel (Eq. 3).
// This family streams X and Omega twice per iteration (once per half-step); the
// fused per-pixel-tile kernel (nmf_fused.cu) streams them once and is preferred
// whenever the shape is inside its compiled range.  The generic path is also the
// projection engine (nmf_project = W-type half-steps with H frozen, reading G11).
//
// Thread mappings (K is split over KS lanes of KC components each, KS*KC >= K):
//   H half-step : one (pixel, k-chunk) per thread; loop over frames; W rows are
//                 broadcast from shared memory; S = (WH)[n,p] never leaves registers.
//   W half-step : one (frame, k-chunk) per thread; loop over pixels; H' columns are
//                 broadcast from shared memory; X/Omega tiles are transposed through
//                 shared memory; per-CTA partial sums go to a slab in the workspace.
//   reduce      : fixed-order fp64 sum of the slabs, then W <- W o A / max(B, eps).
#include "nmf_common.cuh"

namespace {

constexpr int GH_THREADS = 128;  // H half-step CTA size
constexpr int GW_TP = 32;        // pixels per staged chunk in the W half-step
constexpr unsigned FULL = 0xffffffffu;

// ---------------------------------------------------------------------------
// H half-step: H[:,p] <- H[:,p] o W^T(Om o X)[:,p] / W^T(Om o (W H))[:,p]
// ---------------------------------------------------------------------------
template <int KC, int KS>
__global__ void __launch_bounds__(GH_THREADS)
k_h_step(const float* __restrict__ X, const float* __restrict__ Om, const float* __restrict__ W,
         float* __restrict__ H, int N, long long P, int K) {
    constexpr int KT = KC * KS;
    constexpr int PPW = 32 / KS;  // pixels per warp
    extern __shared__ __align__(16) float smem[];  // Ws[N][KT], zero padded
    const int b = blockIdx.y;
    X += (size_t)b * N * P; Om += (size_t)b * N * P; W += (size_t)b * N * K; H += (size_t)b * K * P;
    for (int i = threadIdx.x; i < N * KT; i += GH_THREADS) {
        int n = i / KT, kk = i - n * KT;
        smem[i] = kk < K ? W[(size_t)n * K + kk] : 0.f;
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ks = lane / PPW, pl = lane % PPW;
    const long long p = ((long long)blockIdx.x * (GH_THREADS / 32) + warp) * PPW + pl;
    const bool active = p < P;
    float h[KC], num[KC], den[KC];
#pragma unroll
    for (int j = 0; j < KC; ++j) {
        int k = ks * KC + j;
        h[j] = (active && k < K) ? H[(size_t)k * P + p] : 0.f;
        num[j] = 0.f; den[j] = 0.f;
    }
    const float* wrow = smem + ks * KC;
    const float* xp = X + p;
    const float* op = Om + p;
#pragma unroll 2
    for (int n = 0; n < N; ++n) {
        float om = 0.f, x = 0.f;
        if (active) { om = __ldg(op + (size_t)n * P); x = __ldg(xp + (size_t)n * P); }
        const float4* w4 = reinterpret_cast<const float4*>(wrow + n * KT);
        float wv[KC];
#pragma unroll
        for (int j = 0; j < KC / 4; ++j) {
            float4 t = w4[j];
            wv[4 * j] = t.x; wv[4 * j + 1] = t.y; wv[4 * j + 2] = t.z; wv[4 * j + 3] = t.w;
        }
        float s0 = 0.f, s1 = 0.f;
#pragma unroll
        for (int j = 0; j < KC; j += 2) { s0 = fmaf(wv[j], h[j], s0); s1 = fmaf(wv[j + 1], h[j + 1], s1); }
        float s = s0 + s1;
#pragma unroll
        for (int d = PPW; d < 32; d <<= 1) s += __shfl_xor_sync(FULL, s, d);
        const bool live = om > 0.f;               // Omega == 0: missing datum, skipped (G5)
        const float q = live ? om * x : 0.f;      // (Om o X)[n,p]
        const float r = live ? om * s : 0.f;      // (Om o WH)[n,p]
#pragma unroll
        for (int j = 0; j < KC; ++j) { num[j] = fmaf(wv[j], q, num[j]); den[j] = fmaf(wv[j], r, den[j]); }
    }
    if (active) {
#pragma unroll
        for (int j = 0; j < KC; ++j) {
            int k = ks * KC + j;
            if (k < K) H[(size_t)k * P + p] = (h[j] * num[j]) / fmaxf(den[j], NMF_EPS);
        }
    }
}

// ---------------------------------------------------------------------------
// W half-step, partial sums over a strided set of 32-pixel chunks.
//   A[n,k] = sum_p (Om o X)[n,p] H[k,p],  B[n,k] = sum_p (Om o (W H))[n,p] H[k,p]
// grid: x = pixel partition, y = frame block, z = problem.  slab layout:
//   slab[((z*parts + x)*2 + {A,B}) * N*KT + n*KT + k]
// ---------------------------------------------------------------------------
template <int KC, int KS, bool HAS_OM>
__global__ void __launch_bounds__(512)
k_w_partial(const float* __restrict__ X, const float* __restrict__ Om, const float* __restrict__ W,
            const float* __restrict__ H, float* __restrict__ slab, int N, long long P, int K,
            int NBc) {
    constexpr int KT = KC * KS;
    constexpr int HS = KT + 4;       // hs row stride (floats), keeps float4 alignment
    constexpr int XS = GW_TP + 1;    // xs/os row stride, conflict-free column reads
    extern __shared__ __align__(16) float smem[];
    float* hs = smem;                       // [GW_TP][HS]   H' chunk, transposed
    float* xs = hs + GW_TP * HS;            // [NBc][XS]
    float* os = xs + (size_t)NBc * XS;      // [NBc][XS]
    const int b = blockIdx.z;
    X += (size_t)b * N * P; if (HAS_OM) Om += (size_t)b * N * P;
    W += (size_t)b * N * K; H += (size_t)b * K * P;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int ks = tid % KS, nl = tid / KS;
    const int n0 = blockIdx.y * NBc;
    const int n = n0 + nl;
    const bool valid_n = n < N;
    float w[KC], A[KC], B[KC];
#pragma unroll
    for (int j = 0; j < KC; ++j) {
        int k = ks * KC + j;
        w[j] = (valid_n && k < K) ? W[(size_t)n * K + k] : 0.f;
        A[j] = 0.f; B[j] = 0.f;
    }
    const long long n_chunks = (P + GW_TP - 1) / GW_TP;
    for (long long c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const long long p0 = c * GW_TP;
        __syncthreads();
        for (int i = tid; i < KT * GW_TP; i += nthr) {
            int kk = i / GW_TP, pp = i - kk * GW_TP;
            long long p = p0 + pp;
            hs[pp * HS + kk] = (kk < K && p < P) ? H[(size_t)kk * P + p] : 0.f;
        }
        for (int i = tid; i < NBc * GW_TP; i += nthr) {
            int r = i / GW_TP, pp = i - r * GW_TP;
            long long p = p0 + pp;
            int nn = n0 + r;
            float o = 0.f, x = 0.f;
            if (nn < N && p < P) {
                o = HAS_OM ? Om[(size_t)nn * P + p] : 1.f;
                if (o > 0.f) x = X[(size_t)nn * P + p]; else o = 0.f;   // missing: never read
            }
            xs[r * XS + pp] = x; os[r * XS + pp] = o;
        }
        __syncthreads();
#pragma unroll 1
        for (int pp = 0; pp < GW_TP; ++pp) {
            const float x = xs[nl * XS + pp], o = os[nl * XS + pp];
            const float4* h4 = reinterpret_cast<const float4*>(hs + pp * HS + ks * KC);
            float hv[KC];
#pragma unroll
            for (int j = 0; j < KC / 4; ++j) {
                float4 t = h4[j];
                hv[4 * j] = t.x; hv[4 * j + 1] = t.y; hv[4 * j + 2] = t.z; hv[4 * j + 3] = t.w;
            }
            float s0 = 0.f, s1 = 0.f;
#pragma unroll
            for (int j = 0; j < KC; j += 2) { s0 = fmaf(w[j], hv[j], s0); s1 = fmaf(w[j + 1], hv[j + 1], s1); }
            float s = s0 + s1;
#pragma unroll
            for (int d = 1; d < KS; d <<= 1) s += __shfl_xor_sync(FULL, s, d);
            const bool live = o > 0.f;
            const float q = live ? o * x : 0.f;
            const float r = live ? o * s : 0.f;
#pragma unroll
            for (int j = 0; j < KC; ++j) { A[j] = fmaf(q, hv[j], A[j]); B[j] = fmaf(r, hv[j], B[j]); }
        }
    }
    if (valid_n) {
        float* sa = slab + (((size_t)b * gridDim.x + blockIdx.x) * 2) * (size_t)N * KT + (size_t)n * KT + ks * KC;
        float* sb = sa + (size_t)N * KT;
#pragma unroll
        for (int j = 0; j < KC; j += 4) {
            *reinterpret_cast<float4*>(sa + j) = make_float4(A[j], A[j + 1], A[j + 2], A[j + 3]);
            *reinterpret_cast<float4*>(sb + j) = make_float4(B[j], B[j + 1], B[j + 2], B[j + 3]);
        }
    }
}

// ---------------------------------------------------------------------------
// Fixed-order reduction of the partial slabs (fp64) + W <- W o A / max(B, eps)
// ---------------------------------------------------------------------------
__global__ void k_w_update(const float* __restrict__ slab, float* __restrict__ W, int N, int K,
                           int KT, int parts) {
    const int b = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * K) return;
    const int n = i / K, k = i - n * K;
    const float* s = slab + (size_t)b * parts * 2 * N * KT + (size_t)n * KT + k;
    double a = 0.0, d = 0.0;
    for (int part = 0; part < parts; ++part) {
        a += (double)s[(size_t)(2 * part) * N * KT];
        d += (double)s[(size_t)(2 * part + 1) * N * KT];
    }
    float* w = W + (size_t)b * N * K + i;
    *w = (*w * (float)a) / fmaxf((float)d, NMF_EPS);
}

struct GenericCfg { int kc, ks; };
inline GenericCfg pick_cfg(int K) {
    if (K <= 8) return {8, 1};
    if (K <= 16) return {16, 1};
    if (K <= 32) return {32, 1};
    if (K <= 64) return {32, 2};
    return {32, 4};
}

inline void w_geometry(int rows, int ks, int* nfb, int* NBc, int* threads) {
    int nb_max = 512 / ks;
    *nfb = (rows + nb_max - 1) / nb_max;
    int per = (rows + *nfb - 1) / *nfb;
    *threads = (per * ks + 31) / 32 * 32;
    *NBc = *threads / ks;
}

inline size_t w_smem(int kt, int NBc) {
    return sizeof(float) * ((size_t)GW_TP * (kt + 4) + 2 * (size_t)NBc * (GW_TP + 1));
}

template <int KC, int KS>
int launch_h(nmf_plan* p, const float* X, const float* Om, const float* W, float* H, int batch) {
    const int ppc = GH_THREADS / KS;
    dim3 grid((unsigned)((p->P + ppc - 1) / ppc), batch);
    size_t smem = sizeof(float) * (size_t)p->N * KC * KS;
    static bool attr_done = false;
    if (!attr_done) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_h_step<KC, KS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_done = true;
    }
    k_h_step<KC, KS><<<grid, GH_THREADS, smem, p->stream>>>(X, Om, W, H, p->N, p->P, p->K);
    p->launches++;
    return NMF_OK;
}

template <int KC, int KS>
int launch_w(nmf_plan* p, const float* X, const float* Om, float* W, const float* H, int rows,
             int parts, int batch) {
    int nfb, NBc, threads;
    w_geometry(rows, KS, &nfb, &NBc, &threads);
    size_t smem = w_smem(KC * KS, NBc);
    static bool attr_done = false;
    if (!attr_done) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_w_partial<KC, KS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_w_partial<KC, KS, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
        attr_done = true;
    }
    dim3 grid(parts, nfb, batch);
    float* slab = reinterpret_cast<float*>(p->ws);
    if (Om)
        k_w_partial<KC, KS, true><<<grid, threads, smem, p->stream>>>(X, Om, W, H, slab, rows, p->P, p->K, NBc);
    else
        k_w_partial<KC, KS, false><<<grid, threads, smem, p->stream>>>(X, Om, W, H, slab, rows, p->P, p->K, NBc);
    dim3 g2((rows * p->K + 127) / 128, batch);
    k_w_update<<<g2, 128, 0, p->stream>>>(slab, W, rows, p->K, KC * KS, parts);
    p->launches += 2;
    return NMF_OK;
}

#define DISPATCH_CFG(p, CALL)                                             \
    do {                                                                  \
        if ((p)->g_kc == 8) { CALL(8, 1); }                               \
        else if ((p)->g_kc == 16) { CALL(16, 1); }                        \
        else if ((p)->g_ks == 1) { CALL(32, 1); }                         \
        else if ((p)->g_ks == 2) { CALL(32, 2); }                         \
        else { CALL(32, 4); }                                             \
    } while (0)

int parts_for(const nmf_plan* p, int rows, int batch) {
    int nfb, NBc, threads;
    w_geometry(rows, p->g_ks, &nfb, &NBc, &threads);
    long long n_chunks = (p->P + GW_TP - 1) / GW_TP;
    long long want = (2LL * p->num_sms + (long long)nfb * batch - 1) / ((long long)nfb * batch);
    if (want < 1) want = 1;
    if (want > n_chunks) want = n_chunks;
    return (int)want;
}

}  // namespace

void nmf_generic_configure(nmf_plan* p) {
    GenericCfg c = pick_cfg(p->K);
    p->g_kc = c.kc; p->g_ks = c.ks;
    p->g_parts_fit = parts_for(p, p->N, p->batch);
    p->g_parts_proj = p->max_targets > 0 ? parts_for(p, p->max_targets, 1) : 0;
}

size_t nmf_generic_workspace(const nmf_plan* p) {
    size_t kt = (size_t)p->g_kc * p->g_ks;
    size_t fit = (size_t)p->batch * p->g_parts_fit * 2 * p->N * kt * sizeof(float);
    size_t proj = (size_t)p->g_parts_proj * 2 * p->max_targets * kt * sizeof(float);
    return fit > proj ? fit : proj;
}

int nmf_generic_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters,
                    int batch) {
    const int parts = batch == p->batch ? p->g_parts_fit : parts_for(p, p->N, batch);
    for (int it = 0; it < iters; ++it) {
#define CALL_H(KC, KS) { int rc = launch_h<KC, KS>(p, X, Om, W, H, batch); if (rc) return rc; }
        DISPATCH_CFG(p, CALL_H);
#define CALL_W(KC, KS) { int rc = launch_w<KC, KS>(p, X, Om, W, H, p->N, parts, batch); if (rc) return rc; }
        DISPATCH_CFG(p, CALL_W);
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

int nmf_generic_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C,
                        int M, int iters) {
    const int parts = parts_for(p, M, 1) <= p->g_parts_proj ? parts_for(p, M, 1) : p->g_parts_proj;
    for (int it = 0; it < iters; ++it) {
#define CALL_P(KC, KS) { int rc = launch_w<KC, KS>(p, T, om, C, H, M, parts, 1); if (rc) return rc; }
        DISPATCH_CFG(p, CALL_P);
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

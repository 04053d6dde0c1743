// nmf_generic.cu -- CUDA-core (FFMA) two-kernel path for any N <= 256, K <= 128.
//
// One iteration = H half-step kernel, W half-step partial kernel, fixed-order
// reduction + W update kernel (Eq. 3).
// This family streams X and Omega twice per iteration (once per half-step).  It is
// also the projection engine (nmf_project = W-type half-steps with H frozen, G11).
//
// Register tiling.  K is split over KS lanes (KS a power of two <= 8) of KC components
// each (KS*KC >= K, padded components are exact zeros and stay zero):
//   H half-step : a thread owns 2 adjacent pixels x KC components (h, num, den in
//                 registers); it loops over the frames; the W row chunk comes from
//                 shared memory as a broadcast 128-bit load and is reused for both
//                 pixels and for the three products (6 FFMA per loaded word);
//                 S = (WH)[n,p] is completed across the KS lanes by a shuffle butterfly
//                 and never leaves registers.
//   W half-step : a thread owns NF frames x KC components (W, A, B in registers); it
//                 loops over pixels; the H' column chunk is broadcast from shared memory
//                 and reused for the NF frames; X/Omega tiles are transposed through
//                 shared memory; per-CTA partial sums go to a slab in the workspace.
//   reduce      : fixed-order fp64 sum of the slabs, then W <- W o A / max(B, eps).
// Shared-memory -> register bandwidth (128 B/clk/SM) allows one loaded word per 4 FFMA;
// the tiles above give 6 (H) and 2*NF.. (W) FFMA per broadcast word.
#include "nmf_common.cuh"

namespace {

constexpr int GH_THREADS = 128;  // H half-step CTA size
constexpr int GW_TP = 32;        // pixels per staged chunk in the W half-step
constexpr int GW_XS = GW_TP + 4; // xs/os row stride (floats): 16B-aligned rows, conflict-free float4 reads
constexpr unsigned FULL = 0xffffffffu;

__host__ __device__ constexpr int round4(int v) { return (v + 3) / 4 * 4; }

template <int KC>
__device__ __forceinline__ void load_chunk(float (&dst)[KC], const float* __restrict__ src) {
    // src is 16-byte aligned and holds round4(KC) floats
#pragma unroll
    for (int j = 0; j < KC; j += 4) {
        const float4 t = *reinterpret_cast<const float4*>(src + j);
        dst[j] = t.x;
        if (j + 1 < KC) dst[j + 1] = t.y;
        if (j + 2 < KC) dst[j + 2] = t.z;
        if (j + 3 < KC) dst[j + 3] = t.w;
    }
}

template <int KC>
__device__ __forceinline__ float dot_chunk(const float (&a)[KC], const float (&b)[KC]) {
    float s0 = 0.f, s1 = 0.f;
#pragma unroll
    for (int j = 0; j < KC; ++j) {
        if (j & 1) s1 = fmaf(a[j], b[j], s1); else s0 = fmaf(a[j], b[j], s0);
    }
    return s0 + s1;
}

// ---------------------------------------------------------------------------
// H half-step: H[:,p] <- H[:,p] o W^T(Om o X)[:,p] / W^T(Om o (W H))[:,p]
// thread = (pixel pair, k-chunk kh); lane = kh + KS * pair
// ---------------------------------------------------------------------------
template <int KC>
__global__ void __launch_bounds__(GH_THREADS)
k_h_step(const float* __restrict__ X, const float* __restrict__ Om, const float* __restrict__ W,
         float* __restrict__ H, int N, long long P, int K, int KS) {
    constexpr int KCP = round4(KC);
    extern __shared__ __align__(16) float smem[];  // Ws[N][KS][KCP], zero padded
    const int b = blockIdx.y;
    X += (size_t)b * N * P; Om += (size_t)b * N * P; W += (size_t)b * N * K; H += (size_t)b * K * P;
    const int row = KS * KCP;
    for (int i = threadIdx.x; i < N * row; i += GH_THREADS) {
        const int n = i / row, r = i - n * row, kh = r / KCP, j = r - kh * KCP;
        const int k = kh * KC + j;
        smem[i] = (j < KC && k < K) ? W[(size_t)n * K + k] : 0.f;
    }
    __syncthreads();
    const int kh = threadIdx.x % KS;
    const long long pair = ((long long)blockIdx.x * GH_THREADS + threadIdx.x) / KS;
    const long long p = 2 * pair;
    const bool active = p < P;                    // P is even (P % 4 == 0)
    float h0[KC], h1[KC], num0[KC], num1[KC], den0[KC], den1[KC];
#pragma unroll
    for (int j = 0; j < KC; ++j) {
        const int k = kh * KC + j;
        float2 v = make_float2(0.f, 0.f);
        if (active && k < K) v = *reinterpret_cast<const float2*>(H + (size_t)k * P + p);
        h0[j] = v.x; h1[j] = v.y;
        num0[j] = num1[j] = den0[j] = den1[j] = 0.f;
    }
    const float* wrow = smem + kh * KCP;
    const float* xp = X + p;
    const float* op = Om + p;
#pragma unroll 2
    for (int n = 0; n < N; ++n) {
        float2 om = make_float2(0.f, 0.f), x = make_float2(0.f, 0.f);
        if (active) {
            om = __ldg(reinterpret_cast<const float2*>(op + (size_t)n * P));
            x = __ldg(reinterpret_cast<const float2*>(xp + (size_t)n * P));
        }
        float w[KC];
        load_chunk<KC>(w, wrow + n * row);
        float s0 = dot_chunk<KC>(w, h0);
        float s1 = dot_chunk<KC>(w, h1);
        for (int d = 1; d < KS; d <<= 1) {
            s0 += __shfl_xor_sync(FULL, s0, d);
            s1 += __shfl_xor_sync(FULL, s1, d);
        }
        // Omega == 0: missing datum, skipped (G5); X may be NaN/Inf there
        const float q0 = om.x > 0.f ? om.x * x.x : 0.f, r0 = om.x > 0.f ? om.x * s0 : 0.f;
        const float q1 = om.y > 0.f ? om.y * x.y : 0.f, r1 = om.y > 0.f ? om.y * s1 : 0.f;
#pragma unroll
        for (int j = 0; j < KC; ++j) {
            num0[j] = fmaf(w[j], q0, num0[j]); den0[j] = fmaf(w[j], r0, den0[j]);
            num1[j] = fmaf(w[j], q1, num1[j]); den1[j] = fmaf(w[j], r1, den1[j]);
        }
    }
    if (active) {
#pragma unroll
        for (int j = 0; j < KC; ++j) {
            const int k = kh * KC + j;
            if (k < K) {
                float2 v;
                v.x = (h0[j] * num0[j]) / fmaxf(den0[j], NMF_EPS);
                v.y = (h1[j] * num1[j]) / fmaxf(den1[j], NMF_EPS);
                *reinterpret_cast<float2*>(H + (size_t)k * P + p) = v;
            }
        }
    }
}

// ---------------------------------------------------------------------------
// W half-step, partial sums over a strided set of 32-pixel chunks.
//   A[n,k] = sum_p (Om o X)[n,p] H[k,p],  B[n,k] = sum_p (Om o (W H))[n,p] H[k,p]
// thread = (group of NF frames, k-chunk kh); tid = kh + KS * group
// grid: x = pixel partition, y = frame block, z = problem.  slab layout:
//   slab[((z*parts + x)*2 + {A,B}) * N*KT + n*KT + k],  KT = KS*KC
// ---------------------------------------------------------------------------
template <int KC> __host__ __device__ constexpr int w_max_threads() { return KC > 13 ? 256 : 512; }

template <int KC, int NF, bool HAS_OM>
__global__ void __launch_bounds__(w_max_threads<KC>())
k_w_partial(const float* __restrict__ X, const float* __restrict__ Om, const float* __restrict__ W,
            const float* __restrict__ H, float* __restrict__ slab, int N, long long P, int K,
            int KS, int NBc) {
    constexpr int KCP = round4(KC);
    extern __shared__ __align__(16) float smem[];
    const int hrow = KS * KCP;
    float* hs = smem;                         // [GW_TP][KS][KCP]  H' chunk, transposed
    float* xs = hs + GW_TP * hrow;            // [NBc][GW_XS]
    float* os = xs + (size_t)NBc * GW_XS;     // [NBc][GW_XS]
    const int b = blockIdx.z;
    X += (size_t)b * N * P; if (HAS_OM) Om += (size_t)b * N * P;
    W += (size_t)b * N * K; H += (size_t)b * K * P;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int kh = tid % KS, grp = tid / KS;
    const int n0 = blockIdx.y * NBc;          // first frame of this CTA
    const int KT = KS * KC;
    float w[NF][KC], A[NF][KC], B[NF][KC];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        const int n = n0 + grp * NF + f;
#pragma unroll
        for (int j = 0; j < KC; ++j) {
            const int k = kh * KC + j;
            w[f][j] = (grp * NF + f < NBc && n < N && k < K) ? W[(size_t)n * K + k] : 0.f;
            A[f][j] = 0.f; B[f][j] = 0.f;
        }
    }
    const long long n_chunks = (P + GW_TP - 1) / GW_TP;
    const int xrow = min(grp * NF, NBc - NF);     // clamp idle threads onto valid smem rows
    for (long long c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const long long p0 = c * GW_TP;
        __syncthreads();
        for (int i = tid; i < GW_TP * hrow; i += nthr) {
            // i -> (kh', j, pp) with pp fastest so global reads are coalesced along pixels
            const int pp = i % GW_TP, r = i / GW_TP, khh = r / KCP, j = r - khh * KCP;
            const int k = khh * KC + j;
            const long long p = p0 + pp;
            hs[pp * hrow + r] = (j < KC && k < K && p < P) ? H[(size_t)k * P + p] : 0.f;
        }
        for (int i = tid; i < NBc * GW_TP; i += nthr) {
            const int r = i / GW_TP, pp = i - r * GW_TP;
            const long long p = p0 + pp;
            const int nn = n0 + r;
            float o = 0.f, x = 0.f;
            if (nn < N && p < P) {
                o = HAS_OM ? Om[(size_t)nn * P + p] : 1.f;
                if (o > 0.f) x = X[(size_t)nn * P + p]; else o = 0.f;   // missing: never read
            }
            xs[r * GW_XS + pp] = x; os[r * GW_XS + pp] = o;
        }
        __syncthreads();
#pragma unroll 1
        for (int p4 = 0; p4 < GW_TP; p4 += 4) {
            float xv[NF][4], ov[NF][4];
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const float4 tx = *reinterpret_cast<const float4*>(xs + (xrow + f) * GW_XS + p4);
                const float4 to = *reinterpret_cast<const float4*>(os + (xrow + f) * GW_XS + p4);
                xv[f][0] = tx.x; xv[f][1] = tx.y; xv[f][2] = tx.z; xv[f][3] = tx.w;
                ov[f][0] = to.x; ov[f][1] = to.y; ov[f][2] = to.z; ov[f][3] = to.w;
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                float hv[KC];
                load_chunk<KC>(hv, hs + (p4 + u) * hrow + kh * KCP);
                float s[NF];
#pragma unroll
                for (int f = 0; f < NF; ++f) s[f] = dot_chunk<KC>(w[f], hv);
                for (int d = 1; d < KS; d <<= 1) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) s[f] += __shfl_xor_sync(FULL, s[f], d);
                }
#pragma unroll
                for (int f = 0; f < NF; ++f) {
                    const float o = ov[f][u];
                    const float q = o * xv[f][u];                 // x was zeroed where o == 0
                    const float r = o > 0.f ? o * s[f] : 0.f;
#pragma unroll
                    for (int j = 0; j < KC; ++j) { A[f][j] = fmaf(q, hv[j], A[f][j]); B[f][j] = fmaf(r, hv[j], B[f][j]); }
                }
            }
        }
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        const int n = n0 + grp * NF + f;
        if (grp * NF + f < NBc && n < N) {
            float* sa = slab + (((size_t)b * gridDim.x + blockIdx.x) * 2) * (size_t)N * KT + (size_t)n * KT + kh * KC;
            float* sb = sa + (size_t)N * KT;
#pragma unroll
            for (int j = 0; j < KC; ++j) { sa[j] = A[f][j]; sb[j] = B[f][j]; }
        }
    }
}

// ---------------------------------------------------------------------------
// Fixed-order reduction of the partial slabs (fp64) + W <- W o A / max(B, eps)
// ---------------------------------------------------------------------------
// 256 threads = 32 part lanes x 8 elements: lane q sums the parts q, q + 32, ... in order (independent loads, at most
// five per thread for 148 slabs), the 32 partial sums are then added in lane order -- a fixed association, so the
// result is bitwise reproducible.
constexpr int WU_E = 8, WU_Q = 32;
__global__ void __launch_bounds__(WU_E * WU_Q)
k_w_update(const float* __restrict__ slab, float* __restrict__ W, int N, int K, int KT, int parts) {
    __shared__ double sa[WU_Q][WU_E], sd[WU_Q][WU_E];
    const int b = blockIdx.y;
    const int e = threadIdx.x % WU_E, q = threadIdx.x / WU_E;
    const int i = blockIdx.x * WU_E + e;
    const bool ok = i < N * K;
    const int n = ok ? i / K : 0, k = ok ? i - n * K : 0;
    const size_t stride = (size_t)2 * N * KT;
    const float* s = slab + (size_t)b * parts * stride + (size_t)n * KT + k;
    double a = 0.0, d = 0.0;
    if (ok) {
#pragma unroll 5
        for (int part = q; part < parts; part += WU_Q) {
            a += (double)s[(size_t)part * stride];
            d += (double)s[(size_t)part * stride + (size_t)N * KT];
        }
    }
    sa[q][e] = a; sd[q][e] = d;
    __syncthreads();
    if (q == 0 && ok) {
#pragma unroll
        for (int r = 1; r < WU_Q; ++r) { a += sa[r][e]; d += sd[r][e]; }
        float* w = W + (size_t)b * N * K + i;
        *w = (*w * (float)a) / fmaxf((float)d, NMF_EPS);
    }
}

// ---- host-side geometry -----------------------------------------------------
struct GenericCfg { int kc, ks; };
// pick the (KC, KS) with KC in the compiled set, KS a power of two, least padding
inline GenericCfg pick_cfg(int K) {
    static const int kcs[] = {4, 8, 10, 13, 16};
    GenericCfg best{16, 8};
    int best_pad = 1 << 30;
    for (int ks = 1; ks <= 8; ks <<= 1)
        for (int kc : kcs) {
            int pad = kc * ks - K;
            if (pad < 0) continue;
            // prefer less padding, then fewer lanes (less shuffle work)
            if (pad < best_pad) { best_pad = pad; best = {kc, ks}; }
        }
    return best;
}

constexpr int W_NF = 2;   // frames per thread in the W half-step

constexpr size_t GW_SMEM_MAX = 160 * 1024;   // opt-in dynamic shared memory of k_w_partial

inline void w_geometry(int rows, int kc, int ks, int* nfb, int* NBc, int* threads) {
    // NBc frames per CTA, (NBc / NF) * KS threads, at most 512 (256 for KC = 16) threads, and the staged X / Omega
    // rows (2 NBc rows of GW_XS floats beside the H' chunk) must fit the opt-in shared memory: with ks = 1 the
    // thread limit alone allows 1024 frames per CTA = 288 KB (projection of many frames at K <= 13)
    int nb_max = (kc > 13 ? 256 : 512) / ks * W_NF;
    const int nb_smem = (int)((GW_SMEM_MAX / sizeof(float) - (size_t)GW_TP * ks * round4(kc)) / (2 * GW_XS)) / W_NF * W_NF;
    if (nb_max > nb_smem) nb_max = nb_smem;
    *nfb = (rows + nb_max - 1) / nb_max;
    int per = (rows + *nfb - 1) / *nfb;
    per = (per + W_NF - 1) / W_NF * W_NF;
    *threads = ((per / W_NF) * ks + 31) / 32 * 32;
    *NBc = per;
}

inline size_t w_smem(int kc, int ks, int NBc) {
    return sizeof(float) * ((size_t)GW_TP * ks * round4(kc) + 2 * (size_t)NBc * GW_XS);
}

template <int KC>
int launch_h(nmf_plan* p, const float* X, const float* Om, const float* W, float* H, int batch) {
    const int KS = p->g_ks;
    const long long pairs_per_cta = GH_THREADS / KS;
    dim3 grid((unsigned)((p->P / 2 + pairs_per_cta - 1) / pairs_per_cta), batch);
    size_t smem = sizeof(float) * (size_t)p->N * KS * round4(KC);
    static bool attr_done[NMF_MAX_DEVICES] = {};   // function attributes are per device
    if (!attr_done[p->device]) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_h_step<KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_done[p->device] = true;
    }
    k_h_step<KC><<<grid, GH_THREADS, smem, p->stream>>>(X, Om, W, H, p->N, p->P, p->K, KS);
    p->launches++;
    return NMF_OK;
}

template <int KC>
int launch_w(nmf_plan* p, const float* X, const float* Om, float* W, const float* H, int rows,
             int parts, int batch) {
    const int KS = p->g_ks;
    int nfb, NBc, threads;
    w_geometry(rows, KC, KS, &nfb, &NBc, &threads);
    size_t smem = w_smem(KC, KS, NBc);
    if (smem > GW_SMEM_MAX) return NMF_ERR_UNSUPPORTED;       // (w_geometry caps NBc so that this cannot happen)
    static bool attr_done[NMF_MAX_DEVICES] = {};   // function attributes are per device
    if (!attr_done[p->device]) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_w_partial<KC, W_NF, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GW_SMEM_MAX));
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_w_partial<KC, W_NF, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GW_SMEM_MAX));
        attr_done[p->device] = true;
    }
    dim3 grid(parts, nfb, batch);
    float* slab = reinterpret_cast<float*>(p->ws);
    if (Om)
        k_w_partial<KC, W_NF, true><<<grid, threads, smem, p->stream>>>(X, Om, W, H, slab, rows, p->P, p->K, KS, NBc);
    else
        k_w_partial<KC, W_NF, false><<<grid, threads, smem, p->stream>>>(X, Om, W, H, slab, rows, p->P, p->K, KS, NBc);
    NMF_CUDA_TRY(p, cudaGetLastError());           // a failed launch must not let the update read an unwritten slab
    p->launches++;
    dim3 g2((rows * p->K + WU_E - 1) / WU_E, batch);
    k_w_update<<<g2, WU_E * WU_Q, 0, p->stream>>>(slab, W, rows, p->K, KC * KS, parts);
    p->launches++;
    return NMF_OK;
}

#define DISPATCH_KC(p, CALL)                                 \
    do {                                                     \
        switch ((p)->g_kc) {                                 \
            case 4: CALL(4); break;                          \
            case 8: CALL(8); break;                          \
            case 10: CALL(10); break;                        \
            case 13: CALL(13); break;                        \
            default: CALL(16); break;                        \
        }                                                    \
    } while (0)

int parts_for(const nmf_plan* p, int rows, int batch) {
    int nfb, NBc, threads;
    w_geometry(rows, p->g_kc, p->g_ks, &nfb, &NBc, &threads);
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
    // projection may be called with any M <= max_targets: size for the worst case
    size_t proj = 0;
    for (int M = 1; M <= p->max_targets; ++M) {
        size_t v = (size_t)parts_for(p, M, 1) * 2 * M * kt * sizeof(float);
        if (v > proj) proj = v;
    }
    return fit > proj ? fit : proj;
}

int nmf_launch_w_update(nmf_plan* p, const float* slab, float* W, int rows, int K, int KT, int parts,
                        int batch) {
    dim3 g2((rows * K + WU_E - 1) / WU_E, batch);
    k_w_update<<<g2, WU_E * WU_Q, 0, p->stream>>>(slab, W, rows, K, KT, parts);
    p->launches++;
    return NMF_OK;
}

int nmf_generic_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters,
                    int batch) {
    const int parts = batch == p->batch ? p->g_parts_fit : parts_for(p, p->N, batch);
    int rcl = nmf_run_iterations(p, 10, X, Om, W, H, nullptr, p->N, batch, iters, [&]() -> int {
#define CALL_H(KC) { int rc = launch_h<KC>(p, X, Om, W, H, batch); if (rc) return rc; }
        DISPATCH_KC(p, CALL_H);
#define CALL_W(KC) { int rc = launch_w<KC>(p, X, Om, W, H, p->N, parts, batch); if (rc) return rc; }
        DISPATCH_KC(p, CALL_W);
        return NMF_OK;
    });
    if (rcl) return rcl;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

int nmf_generic_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C,
                        int M, int iters) {
    const int parts = parts_for(p, M, 1);
    int rcl = nmf_run_iterations(p, 11, T, om, C, H, nullptr, M, 1, iters, [&]() -> int {
#define CALL_P(KC) { int rc = launch_w<KC>(p, T, om, C, H, M, parts, 1); if (rc) return rc; }
        DISPATCH_KC(p, CALL_P);
        return NMF_OK;
    });
    if (rcl) return rcl;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

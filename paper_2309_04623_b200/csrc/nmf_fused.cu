// nmf_fused.cu -- fused per-pixel-tile NMF iteration on the FP32 FFMA pipe.
//
// One persistent CTA walks pixel tiles of T = blockDim.x pixels.  Per tile (Eq. 3):
//   H half (thread = one pixel, all K components in registers):
//       for every frame n:  s = W[n,:].h           (a2)   W row broadcast from shared memory
//                           q = Om*X, r = Om*s      (a3)   X, Om straight from global, coalesced
//                           num += W[n,:]*q, den += W[n,:]*r   (a4)
//       h' = h o num / max(den, eps)                (a5)   written to H in place and to a smem tile
//   W half (thread = one frame, all K components in registers), with the new h':
//       for every pixel t:  s' = W[n,:].h'[:,t]     (a6)   h' column broadcast from shared memory
//                           A += q*h'[:,t], B += (Om*s')*h'[:,t]   (a7)
//       X, Om are re-read (L2 hits: the tile was streamed from HBM a moment ago by the same CTA)
//       through cp.async-staged, padded sub-tiles so that a thread walks its own frame row.
//   The per-tile A, B are added to this CTA's slab in the workspace (fixed tile order); the slabs
//   are reduced in fixed order and W updated by nmf_launch_w_update (a8).
// No cross-lane reduction appears in either inner loop: every loaded word of W / h' feeds three
// FFMAs, and the only non-FFMA work per (n, pixel) is the 128-bit broadcast loads (K/4) and ~8
// scalar instructions.  HBM traffic per iteration is the algorithmic 8NP + 8KP bytes.
#include "nmf_common.cuh"

namespace {

constexpr int SUB = 32;          // pixels per cp.async sub-tile of the W half
constexpr int SUBP = SUB + 4;    // padded row stride (floats): conflict-free row-per-thread float4 reads

__host__ __device__ constexpr int round4(int v) { return (v + 3) / 4 * 4; }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, bool valid) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int sz = valid ? 16 : 0;                       // src-size 0: zero-fill, nothing is read
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N_> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N_) : "memory"); }

template <int KC>
__device__ __forceinline__ void lds_row(float (&dst)[KC], const float* __restrict__ src) {
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
__device__ __forceinline__ float dot4(const float (&a)[KC], const float (&b)[KC]) {
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;      // four chains hide the FFMA latency
#pragma unroll
    for (int j = 0; j < KC; ++j) {
        if ((j & 3) == 0) s0 = fmaf(a[j], b[j], s0);
        else if ((j & 3) == 1) s1 = fmaf(a[j], b[j], s1);
        else if ((j & 3) == 2) s2 = fmaf(a[j], b[j], s2);
        else s3 = fmaf(a[j], b[j], s3);
    }
    return (s0 + s1) + (s2 + s3);
}

// issue the cp.async copies of sub-tile `st` of the current tile into stage buffers xs/os
__device__ __forceinline__ void stage_subtile(float* xs, float* os, const float* __restrict__ X,
                                              const float* __restrict__ Om, int N, long long P,
                                              long long p_sub) {
    constexpr int CH = SUB / 4;
    for (int i = threadIdx.x; i < N * CH; i += blockDim.x) {
        const int n = i / CH, c = i - n * CH;
        const long long p = p_sub + 4 * c;
        const bool ok = p < P;                            // P % 4 == 0: a chunk is all in or all out
        const size_t g = (size_t)n * P + (ok ? p : 0);
        cp_async16(xs + n * SUBP + 4 * c, X + g, ok);
        cp_async16(os + n * SUBP + 4 * c, Om + g, ok);
    }
    cp_async_commit();
}

template <int KC>
__global__ void __launch_bounds__(256)
k_fused_iter(const float* __restrict__ X, const float* __restrict__ Om, const float* __restrict__ W,
             float* __restrict__ H, float* __restrict__ slab, int N, long long P, int K, int FPW,
             long long n_tiles) {
    constexpr int KCP = round4(KC);
    extern __shared__ __align__(16) float smem[];
    const int T = blockDim.x;
    float* Ws = smem;                                  // [N][KCP]   zero-padded W
    float* Hs = Ws + (size_t)N * KCP;                  // [T][KCP]   h' of the current tile
    float* Xs = Hs + (size_t)T * KCP;                  // [2][N][SUBP]
    float* Os = Xs + 2 * (size_t)N * SUBP;             // [2][N][SUBP]
    const int b = blockIdx.y;
    X += (size_t)b * N * P; Om += (size_t)b * N * P; W += (size_t)b * N * K; H += (size_t)b * K * P;
    slab += ((size_t)b * gridDim.x + blockIdx.x) * 2 * (size_t)N * KCP;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    for (int i = tid; i < N * KCP; i += T) {
        const int n = i / KCP, j = i - n * KCP;
        Ws[i] = j < K ? W[(size_t)n * K + j] : 0.f;
    }
    // W-half ownership: warp w owns frames [w*FPW, w*FPW+FPW), lane = frame within the warp
    const int wn = warp * FPW + lane;
    const bool w_active = lane < FPW && wn < N;
    const int wn_c = w_active ? wn : 0;
    const int n_sub = (T + SUB - 1) / SUB;
    bool first = true;
    __syncthreads();

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long p0 = tile * T;
        // sub-tile 0 of the W half travels while the H half computes
        stage_subtile(Xs, Os, X, Om, N, P, p0);

        // ------------------------------ H half ------------------------------
        {
            const long long p = p0 + tid;
            const bool active = p < P;
            const long long pc = active ? p : P - 1;
            float h[KC], num[KC], den[KC];
#pragma unroll
            for (int j = 0; j < KC; ++j) {
                h[j] = j < K ? H[(size_t)j * P + pc] : 0.f;
                num[j] = 0.f; den[j] = 0.f;
            }
            const float* xp = X + pc;
            const float* op = Om + pc;
            float xv[4], ov[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int nn = min(u, N - 1);
                xv[u] = __ldg(xp + (size_t)nn * P); ov[u] = __ldg(op + (size_t)nn * P);
            }
            for (int n0 = 0; n0 < N; n0 += 4) {
                float xn[4], on[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {               // prefetch the next four frames
                    const int nn = min(n0 + 4 + u, N - 1);
                    xn[u] = __ldg(xp + (size_t)nn * P); on[u] = __ldg(op + (size_t)nn * P);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (n0 + u < N) {
                        float w[KC];
                        lds_row<KC>(w, Ws + (n0 + u) * KCP);
                        const float s = dot4<KC>(w, h);
                        const float o = ov[u];
                        // Omega == 0: missing datum, skipped (G5); X may be NaN/Inf there
                        const float q = o > 0.f ? o * xv[u] : 0.f;
                        const float r = o > 0.f ? o * s : 0.f;
#pragma unroll
                        for (int j = 0; j < KC; ++j) {
                            num[j] = fmaf(w[j], q, num[j]);
                            den[j] = fmaf(w[j], r, den[j]);
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) { xv[u] = xn[u]; ov[u] = on[u]; }
            }
            float hn[KCP];
#pragma unroll
            for (int j = 0; j < KCP; ++j) {
                float v = 0.f;
                if (j < KC) {
                    v = (h[j] * num[j]) / fmaxf(den[j], NMF_EPS);
                    if (!active) v = 0.f;
                    if (active && j < K) H[(size_t)j * P + p] = v;
                }
                hn[j] = v;
            }
            __syncthreads();        // every W-half reader of the previous tile's Hs is done
#pragma unroll
            for (int j = 0; j < KCP; j += 4)
                *reinterpret_cast<float4*>(Hs + (size_t)tid * KCP + j) = make_float4(hn[j], hn[j + 1], hn[j + 2], hn[j + 3]);
        }

        // ------------------------------ W half ------------------------------
        {
            float wr[KC], A[KC], B[KC];
            lds_row<KC>(wr, Ws + (size_t)wn_c * KCP);
#pragma unroll
            for (int j = 0; j < KC; ++j) { A[j] = 0.f; B[j] = 0.f; }
            for (int st = 0; st < n_sub; ++st) {
                const int cur = st & 1;
                if (st + 1 < n_sub) {
                    stage_subtile(Xs + (size_t)(cur ^ 1) * N * SUBP, Os + (size_t)(cur ^ 1) * N * SUBP, X, Om, N, P,
                                  p0 + (long long)(st + 1) * SUB);
                    cp_async_wait<1>();
                } else {
                    cp_async_wait<0>();
                }
                __syncthreads();    // stage `cur` (and, for st == 0, the Hs tile) visible to everyone
                if (w_active) {
                    const float* xrow = Xs + (size_t)cur * N * SUBP + (size_t)wn * SUBP;
                    const float* orow = Os + (size_t)cur * N * SUBP + (size_t)wn * SUBP;
                    const int t_lim = min(SUB, T - st * SUB);
#pragma unroll 1
                    for (int t4 = 0; t4 < t_lim; t4 += 4) {
                        const float4 x4 = *reinterpret_cast<const float4*>(xrow + t4);
                        const float4 o4 = *reinterpret_cast<const float4*>(orow + t4);
                        const float xa[4] = {x4.x, x4.y, x4.z, x4.w};
                        const float oa[4] = {o4.x, o4.y, o4.z, o4.w};
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            float hv[KC];
                            lds_row<KC>(hv, Hs + (size_t)(st * SUB + t4 + u) * KCP);
                            const float s = dot4<KC>(wr, hv);
                            const float o = oa[u];
                            const float q = o > 0.f ? o * xa[u] : 0.f;
                            const float r = o > 0.f ? o * s : 0.f;
#pragma unroll
                            for (int j = 0; j < KC; ++j) {
                                A[j] = fmaf(q, hv[j], A[j]);
                                B[j] = fmaf(r, hv[j], B[j]);
                            }
                        }
                    }
                }
                __syncthreads();    // stage `cur` may be overwritten by the copy issued next round
            }
            // per-tile partial -> this CTA's slab (fixed tile order => deterministic)
            if (w_active) {
                float* sa = slab + (size_t)wn * KCP;
                float* sb = sa + (size_t)N * KCP;
#pragma unroll
                for (int j = 0; j < KC; ++j) {
                    if (first) { sa[j] = A[j]; sb[j] = B[j]; }
                    else { sa[j] += A[j]; sb[j] += B[j]; }
                }
            }
            first = false;
        }
    }
    // a CTA that had no tile still owns a slab: it must read as zero
    if (first && w_active) {
        float* sa = slab + (size_t)wn * KCP;
        float* sb = sa + (size_t)N * KCP;
#pragma unroll
        for (int j = 0; j < KC; ++j) { sa[j] = 0.f; sb[j] = 0.f; }
    }
}

// ---- host side -----------------------------------------------------------------
const int kKC[] = {1, 2, 3, 5, 8, 10, 13, 16, 20, 25, 30, 40, 50};

int pick_kc(int K) {
    for (int kc : kKC) if (kc >= K) return kc;
    return 0;
}

size_t fused_smem(int N, int T, int kc) {
    return sizeof(float) * ((size_t)N * round4(kc) + (size_t)T * round4(kc) + 4 * (size_t)N * SUBP);
}

template <int KC>
int launch(nmf_plan* p, const float* X, const float* Om, const float* W, float* H, int batch) {
    const int T = p->f_threads;
    const size_t smem = fused_smem(p->N, T, KC);
    static bool attr_done[NMF_MAX_DEVICES] = {};   // the opt-in shared-memory size is a per-device function attribute
    if (!attr_done[p->device]) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_fused_iter<KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        attr_done[p->device] = true;
    }
    const long long n_tiles = (p->P + T - 1) / T;
    dim3 grid(p->f_ctas, batch);
    k_fused_iter<KC><<<grid, T, smem, p->stream>>>(X, Om, W, H, reinterpret_cast<float*>(p->ws), p->N, p->P, p->K,
                                                   p->f_fpw, n_tiles);
    p->launches++;
    return NMF_OK;
}

template <int KC>
int occupancy(int T, size_t smem) {
    int nb = 0;
    if (cudaFuncSetAttribute(k_fused_iter<KC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_fused_iter<KC>, T, smem) != cudaSuccess) return 0;
    return nb;
}

#define FUSED_DISPATCH(kc, CALL)                                                        \
    switch (kc) {                                                                       \
        case 1: CALL(1); break;   case 2: CALL(2); break;   case 3: CALL(3); break;     \
        case 5: CALL(5); break;   case 8: CALL(8); break;   case 10: CALL(10); break;   \
        case 13: CALL(13); break; case 16: CALL(16); break; case 20: CALL(20); break;   \
        case 25: CALL(25); break; case 30: CALL(30); break; case 40: CALL(40); break;   \
        case 50: CALL(50); break; default: break;                                       \
    }

}  // namespace

void nmf_fused_configure(nmf_plan* p) {
    p->f_kp = 0; p->f_ctas = 0; p->f_threads = 0; p->f_fpw = 0;
    const int kc = pick_kc(p->K);
    if (!kc) return;
    // CTA size: one thread per frame in the W half, rounded up to whole warps (<= 256)
    int T = (p->N + 31) / 32 * 32;
    if (T > 256) return;
    if (T == 96) T = 128;                       // keep the four SM sub-partitions evenly loaded
    if (T > 128 && T < 256) T = 256;
    const int warps = T / 32;
    const int fpw = (p->N + warps - 1) / warps;
    const size_t smem = fused_smem(p->N, T, kc);
    if (smem > 227 * 1024) return;
    int occ = 0;
#define OCC(KC) occ = occupancy<KC>(T, smem)
    FUSED_DISPATCH(kc, OCC);
    if (occ < 1) return;
    const long long n_tiles = (p->P + T - 1) / T;
    long long ctas = (long long)p->num_sms * occ / p->batch;
    if (ctas < 1) ctas = 1;
    if (ctas > n_tiles) ctas = n_tiles;
    // even out the tiles: every CTA gets ceil(n_tiles / ctas) or one fewer
    const long long per = (n_tiles + ctas - 1) / ctas;
    ctas = (n_tiles + per - 1) / per;
    p->f_kp = kc; p->f_ctas = (int)ctas; p->f_threads = T; p->f_fpw = fpw;
}

size_t nmf_fused_workspace(const nmf_plan* p) {
    if (!p->f_kp) return 0;
    return (size_t)p->batch * p->f_ctas * 2 * p->N * round4(p->f_kp) * sizeof(float);
}

bool nmf_fused_available(const nmf_plan* p) { return p->f_kp != 0; }

int nmf_fused_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters, int batch) {
    if (!p->f_kp) return NMF_ERR_UNSUPPORTED;
    const int kcp = round4(p->f_kp);
    int rcl = nmf_run_iterations(p, 20, X, Om, W, H, nullptr, p->N, batch, iters, [&]() -> int {
#define CALL_F(KC) { int rc = launch<KC>(p, X, Om, W, H, batch); if (rc) return rc; }
        FUSED_DISPATCH(p->f_kp, CALL_F);
        return nmf_launch_w_update(p, reinterpret_cast<const float*>(p->ws), W, p->N, p->K, kcp, p->f_ctas, batch);
    });
    if (rcl) return rcl;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

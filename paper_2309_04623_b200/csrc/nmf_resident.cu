// nmf_resident.cu -- ALL iterations of Eq. 3 in ONE cooperative launch, for problems small enough to
// stay on chip: K <= 8, N <= 64, at most one 128-pixel tile per SM (P <= 128 x SMs), one problem.
//
// Such a problem (the "tiny" config: 16 frames x 64^2 px x 5 components) is bound by launches, not by bytes or flops: two
// kernels per iteration, replayed from a CUDA graph, cost 14 us per iteration.  Here CTA c keeps its tile of X and Omega
// in shared memory and its tile of H in REGISTERS (thread = pixel) for the whole fit; per iteration it does the
// H half-step locally, reduces its partial A = Q H'^T, B = R' H'^T over its 128 pixels (shuffles, then the four warps in
// order), writes them to its slab, and meets the other CTAs at ONE grid-wide barrier (a monotonic counter in global
// memory; the launch is cooperative, so all CTAs are resident).  After the barrier every CTA adds the slabs of all CTAs in
// CTA order in fp64 and updates its own copy of W -- the same arithmetic in every CTA, so the copies stay bitwise equal.
// Slabs are double-buffered by iteration parity: a CTA can run at most one barrier ahead of the slowest.
// H and W go back to global memory once, at the end.
#include "nmf_common.cuh"

namespace {

constexpr int RS_PX = 128;                // pixels per CTA = threads per CTA
constexpr int RS_MAXK = 8, RS_MAXN = 64;

struct ResArgs {
    const float* X; const float* Om; float* W; float* H;
    float* slab;                          // [2 parities][ctas][N][2K]
    unsigned int* counter;                // grid barrier: arrivals so far (zeroed before the launch)
    int N, iters; long long P;
};

template <int K>
__global__ void __launch_bounds__(RS_PX, 1)
k_resident(const ResArgs g) {
    extern __shared__ __align__(16) float rs_smem[];
    const int N = g.N;
    float* xs = rs_smem;                  // [N][128]
    float* os = xs + N * RS_PX;           // [N][128]
    float* ws = os + N * RS_PX;           // [N][K]
    float* part = ws + N * K;             // [4 warps][N][2K]
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const long long p = (long long)blockIdx.x * RS_PX + t;
    const bool in = p < g.P;
    for (int n = 0; n < N; ++n) {
        xs[n * RS_PX + t] = in ? g.X[(size_t)n * g.P + p] : 0.f;
        os[n * RS_PX + t] = in ? g.Om[(size_t)n * g.P + p] : 0.f;        // Omega = 0 beyond P: those pixels contribute nothing
    }
    for (int i = t; i < N * K; i += RS_PX) ws[i] = g.W[i];
    float h[K];
#pragma unroll
    for (int k = 0; k < K; ++k) h[k] = in ? g.H[(size_t)k * g.P + p] : 0.f;
    __syncthreads();
    const size_t slab_stride = (size_t)gridDim.x * N * 2 * K;            // one parity

    for (int it = 0; it < g.iters; ++it) {
        // ---------------- H half-step (a1-a5): thread = pixel ----------------
        float num[K], den[K];
#pragma unroll
        for (int k = 0; k < K; ++k) { num[k] = 0.f; den[k] = 0.f; }
        for (int n = 0; n < N; ++n) {
            const float x = xs[n * RS_PX + t], o = os[n * RS_PX + t];
            float sv = 0.f;
#pragma unroll
            for (int k = 0; k < K; ++k) sv = fmaf(ws[n * K + k], h[k], sv);
            const bool live = o > 0.f;
            const float q = live ? o * x : 0.f, r = live ? o * sv : 0.f;
#pragma unroll
            for (int k = 0; k < K; ++k) { num[k] = fmaf(ws[n * K + k], q, num[k]); den[k] = fmaf(ws[n * K + k], r, den[k]); }
        }
#pragma unroll
        for (int k = 0; k < K; ++k) h[k] = (h[k] * num[k]) / fmaxf(den[k], NMF_EPS);
        // ---------------- W half-step partials (a6-a7): sum over the CTA's pixels ----------------
        for (int n = 0; n < N; ++n) {
            const float x = xs[n * RS_PX + t], o = os[n * RS_PX + t];
            float sv = 0.f;
#pragma unroll
            for (int k = 0; k < K; ++k) sv = fmaf(ws[n * K + k], h[k], sv);
            const bool live = o > 0.f;
            const float q = live ? o * x : 0.f, r = live ? o * sv : 0.f;
            float v[2 * K];
#pragma unroll
            for (int k = 0; k < K; ++k) { v[k] = q * h[k]; v[K + k] = r * h[k]; }
#pragma unroll
            for (int m = 16; m > 0; m >>= 1)
#pragma unroll
                for (int k = 0; k < 2 * K; ++k) v[k] += __shfl_xor_sync(0xffffffffu, v[k], m);
            if (lane == 0) {
#pragma unroll
                for (int k = 0; k < 2 * K; ++k) part[(warp * N + n) * 2 * K + k] = v[k];
            }
        }
        __syncthreads();
        float* my = g.slab + (size_t)(it & 1) * slab_stride + (size_t)blockIdx.x * N * 2 * K;
        for (int i = t; i < N * 2 * K; i += RS_PX)
            my[i] = ((part[i] + part[N * 2 * K + i]) + part[2 * N * 2 * K + i]) + part[3 * N * 2 * K + i];
        // ---------------- grid-wide barrier: the CTA's slab stores are ordered before thread 0's release by the CTA
        // barrier, the other CTAs' slabs after its acquire ----------------
        __syncthreads();
        if (t == 0) {
            const unsigned int want = (unsigned int)(it + 1) * gridDim.x;
            unsigned int seen;
            asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(g.counter) : "memory");
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(g.counter) : "memory");
            } while (seen < want);
        }
        __syncthreads();
        // ---------------- a8: every CTA adds all slabs in CTA order (fp64) and updates its copy of W ----------------
        const float* all = g.slab + (size_t)(it & 1) * slab_stride;
        for (int i = t; i < N * K; i += RS_PX) {
            const int n = i / K, k = i - n * K;
            double a = 0.0, bsum = 0.0;
#pragma unroll 8
            for (unsigned int c = 0; c < gridDim.x; ++c) {
                a += (double)__ldcg(all + ((size_t)c * N + n) * 2 * K + k);
                bsum += (double)__ldcg(all + ((size_t)c * N + n) * 2 * K + K + k);
            }
            ws[i] = (ws[i] * (float)a) / fmaxf((float)bsum, NMF_EPS);
        }
        __syncthreads();
    }
    if (in) {
#pragma unroll
        for (int k = 0; k < K; ++k) g.H[(size_t)k * g.P + p] = h[k];
    }
    if (blockIdx.x == 0)
        for (int i = t; i < N * K; i += RS_PX) g.W[i] = ws[i];
}

inline size_t res_smem(int N, int K) { return sizeof(float) * ((size_t)2 * N * RS_PX + (size_t)N * K + (size_t)4 * N * 2 * K); }
inline int res_ctas(const nmf_plan* p) { return (int)((p->P + RS_PX - 1) / RS_PX); }
inline size_t res_slab_bytes(const nmf_plan* p) { return nmf_align_up((size_t)2 * res_ctas(p) * p->N * 2 * p->K * sizeof(float), 256); }

template <int K>
cudaError_t launch_resident(ResArgs& a, int ctas, size_t smem, cudaStream_t st, int device) {
    static bool done[NMF_MAX_DEVICES] = {};               // the opt-in shared-memory size is a per-device attribute
    if (!done[device]) {
        cudaError_t e = cudaFuncSetAttribute(k_resident<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        done[device] = true;
    }
    void* args[] = {&a};
    return cudaLaunchCooperativeKernel(reinterpret_cast<void*>(k_resident<K>), dim3(ctas), dim3(RS_PX), args, smem, st);
}

}  // namespace

void nmf_resident_configure(nmf_plan* p) {
    p->rs_ok = false;
    if (p->K > RS_MAXK || p->N > RS_MAXN || p->batch != 1) return;
    if (res_ctas(p) > p->num_sms) return;                 // every CTA must be resident: one per SM
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, p->device) != cudaSuccess || !coop) return;
    p->rs_ok = true;
}

bool nmf_resident_available(const nmf_plan* p) { return p->rs_ok; }

// slabs of both parities + the barrier counter
size_t nmf_resident_workspace(const nmf_plan* p) { return p->rs_ok ? res_slab_bytes(p) + 256 : 0; }

int nmf_resident_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters) {
    if (!p->rs_ok) return NMF_ERR_UNSUPPORTED;
    ResArgs a{};
    a.X = X; a.Om = Om; a.W = W; a.H = H; a.N = p->N; a.P = p->P; a.iters = iters;
    a.slab = reinterpret_cast<float*>(p->ws);
    a.counter = reinterpret_cast<unsigned int*>(static_cast<char*>(p->ws) + res_slab_bytes(p));
    NMF_CUDA_TRY(p, cudaMemsetAsync(a.counter, 0, sizeof(unsigned int), p->stream));
    const int ctas = res_ctas(p), K = p->K;
    const size_t smem = res_smem(p->N, K);
    cudaError_t e = K == 1 ? launch_resident<1>(a, ctas, smem, p->stream, p->device) : K == 2 ? launch_resident<2>(a, ctas, smem, p->stream, p->device) :
                    K == 3 ? launch_resident<3>(a, ctas, smem, p->stream, p->device) : K == 4 ? launch_resident<4>(a, ctas, smem, p->stream, p->device) :
                    K == 5 ? launch_resident<5>(a, ctas, smem, p->stream, p->device) : K == 6 ? launch_resident<6>(a, ctas, smem, p->stream, p->device) :
                    K == 7 ? launch_resident<7>(a, ctas, smem, p->stream, p->device) : launch_resident<8>(a, ctas, smem, p->stream, p->device);
    NMF_CUDA_TRY(p, e);
    p->launches += 1;
    return NMF_OK;
}

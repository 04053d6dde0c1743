// nmf_stream.cu -- one iteration of Eq. 3 for FEW components (K <= 8) as ONE streaming FP32 kernel.
//
// With K <= 8 an element (frame, pixel) costs 6K flops per half-step: less than the 13 instructions the tensor-core
// kernels spend on splitting q and r into BF16 pieces, so the contractions stay on the FFMA pipe and the kernel is
// bound by HBM: X and Omega cross it ONCE per iteration.  A persistent CTA (512 threads) takes pixel tiles of 32:
// TMA lands the tile's [N frames][32 px] of X and of Omega (128-byte rows, 128-byte swizzle) and its [K][32 px] of H in
// one of NS stages of shared memory, and both half-steps read them from there:
//   H half-step (a1-a5)  lane = pixel, warp w takes frames w, w + 16, ...: s = W[n,:].h, q = Omega o x, r = Omega o s,
//                        num += W[n,:] q, den += W[n,:] r; the 16 warps' partial sums are added in warp order through
//                        shared memory; h' = h num / max(den, eps) -> global H and shared memory.
//   W half-step (a6-a7)  thread = (frames j and j + ceil(N/2), 8 of the 32 pixels): s' = W[n,:].h', A[n,:] += q h',
//                        B[n,:] += r' h' in registers over ALL tiles of the CTA; at the end the four threads of a
//                        frame pair add up (shuffles) and write the CTA's slab [2][N][K].
//   k_w_update_stream    fixed-order fp64 reduction of the slabs + W <- W o A / max(B, eps)   (a8)
// Select semantics (entries with Omega == 0 never touch X), plain IEEE division: bitwise reproducible, exact under
// power-of-two scaling.  Rows of a stage are addressed through the swizzle: 16-byte chunk c of row n lies at c ^ (n & 7).
#include <cuda.h>
#include "nmf_common.cuh"
#include "nmf_tc.cuh"

namespace {
using namespace tc;

constexpr int ST_GROUPS = 2, ST_GWARPS = 8, ST_GTHREADS = 32 * ST_GWARPS;       // two groups of eight compute warps
constexpr int ST_CWARPS = ST_GROUPS * ST_GWARPS, ST_THREADS = 32 * (ST_CWARPS + 1), ST_PX = 32;   // + one TMA producer warp
constexpr int ST_MAXK = 8;
constexpr int ST_MAX_STAGES = 4;
// iterations per call from which the tile-major copy of X, Omega pays: it costs about two iterations' time and saves 30 %
// per iteration at K = 1 (HBM-bound), 13 % at K = 3, but only 1-3 % from K = 4 (issue-bound)
inline int tiled_min_iters(int K) { return K <= 2 ? 8 : K == 3 ? 16 : 64; }
constexpr size_t ST_SMEM_MAX = 227 * 1024;

struct StreamArgs {
    CUtensorMap mX, mO;        // X, Om [B*N, P]: box [N frames][32 px], 128-byte swizzle
    CUtensorMap mH;            // H [B*K, P]: box [K][32 px]
    const float* W; float* H; float* slab;
    const float* Xt; const float* Ot;   // tile-major copies of X and Omega (k_tile_major), or null: read X, Omega through mX, mO
    int N, NS; long long P; long long n_tiles;
    int xbytes;                // bytes of one X (or Omega) box, rounded up to 1024
    int stage_bytes;
};

// 1-D bulk copy global -> shared memory, completing on an mbarrier (bytes % 16 == 0, both addresses 16-byte aligned)
__device__ __forceinline__ void bulk_load(uint32_t smem_dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_dst), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// Tile-major copy of X (z even) or Omega (z odd) of problem z / 2: out[tile][n][32 px] with the 16-byte chunks of a row
// stored where the 128-byte swizzle puts them (chunk c of row n at c ^ (n & 7)), pixels beyond P as zeros -- byte for
// byte the shared-memory image of a stage, so that a tile is ONE contiguous block of N x 128 bytes.
// Why: with the caller's [N, P] layout every row of a tile is its own 128-byte request 4P bytes from the next (4 MB =
// two pages at P = 1024^2) and the streaming kernel reached 4.4 TB/s; the same bytes with rows 256 KB apart (16 problems
// of 65536 pixels) ran at 5.85 TB/s.  One pass of 2 x 8NP bytes per nmf_fit call, worth it from a few iterations up.
__global__ void __launch_bounds__(256)
k_tile_major(const float* __restrict__ X, const float* __restrict__ Om, float* __restrict__ Xt, float* __restrict__ Ot,
             int N, long long P, long long n_tiles) {
    const int n = blockIdx.y, b = blockIdx.z >> 1;
    const float* __restrict__ src = ((blockIdx.z & 1) ? Om : X) + ((size_t)b * N + n) * P;
    float* __restrict__ dst = ((blockIdx.z & 1) ? Ot : Xt) + (size_t)b * n_tiles * N * ST_PX;
    const long long ch = (long long)blockIdx.x * 256 + threadIdx.x;      // 16-byte chunk of the row
    if (ch >= n_tiles * 8) return;
    const long long tile = ch >> 3;
    const int c = (int)(ch & 7);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (4 * ch < P) v = __ldg(reinterpret_cast<const float4*>(src + 4 * ch));     // P % 4 == 0
    *reinterpret_cast<float4*>(dst + ((size_t)tile * N + n) * ST_PX + 4 * (c ^ (n & 7))) = v;
}

// Tiles alternate between the two groups (tile i of the CTA -> group i & 1), so that one group's H half-step overlaps
// the other's W half-step; the stages form one ring filled by the producer warp.  An mbarrier wait tests a phase
// PARITY: every compute warp therefore waits for EVERY tile's "full" barrier in ring order and arrives on its "empty"
// barrier (count = all compute warps) -- for the other group's tiles without touching the data -- so no waiter is ever
// two phases away from the barrier it tests.
template <int K>
__global__ void __launch_bounds__(ST_THREADS, 1)
k_stream(const __grid_constant__ StreamArgs g) {
    constexpr int KP4 = (K + 3) / 4 * 4;
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, NH = (N + 1) / 2;
    unsigned char* stages = smem;
    float* Ws = reinterpret_cast<float*>(smem + (size_t)g.NS * g.stage_bytes);     // [N][KP4]
    float* red0 = Ws + (size_t)N * KP4;                                            // [group][8 warps][2K][32]
    float* hn0 = red0 + ST_GROUPS * ST_GWARPS * 2 * K * ST_PX;                     // [group][K][32] new h
    uint64_t* full = reinterpret_cast<uint64_t*>(hn0 + ST_GROUPS * K * ST_PX);     // [NS]
    uint64_t* empty = full + ST_MAX_STAGES;                                        // [NS]
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y;
    const float* __restrict__ Wg = g.W + (size_t)b * N * K;
    float* __restrict__ Hg = g.H + (size_t)b * K * g.P;
    // A CTA takes PAIRS of adjacent tiles (pair q = blockIdx.x + i gridDim.x, tiles 2q and 2q + 1, one per group): the two
    // 128-byte segments of a row are requested close together in time.  gridDim.x <= number of pairs.
    const long long n_pairs = (g.n_tiles + 1) / 2;
    const uint32_t my_pairs = (uint32_t)((n_pairs - 1 - blockIdx.x) / gridDim.x) + 1u;
    const bool last_half = (g.n_tiles & 1) && (blockIdx.x + (long long)(my_pairs - 1) * gridDim.x == n_pairs - 1);
    const uint32_t n_my = 2u * my_pairs - (last_half ? 1u : 0u);
    auto tile_px = [&](uint32_t i) -> long long { return ((blockIdx.x + (long long)(i >> 1) * gridDim.x) * 2 + (i & 1u)) * ST_PX; };
    const uint32_t NS = (uint32_t)g.NS;

    if (tid == 0) {
        for (uint32_t s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], ST_CWARPS); }
        mbar_fence_init();
        tma_prefetch_desc(&g.mX); tma_prefetch_desc(&g.mO); tma_prefetch_desc(&g.mH);
    }
    for (int i = tid; i < N * KP4; i += ST_THREADS) {
        const int n = i / KP4, k = i - n * KP4;
        Ws[i] = k < K ? Wg[(size_t)n * K + k] : 0.f;
    }
    __syncthreads();

    if (warp == ST_CWARPS) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            const uint32_t tx_bytes = (uint32_t)(2 * N * 128 + K * 128);
            for (uint32_t i = 0; i < n_my; ++i) {
                const uint32_t s = i % NS, u = i / NS;
                if (u > 0) mbar_wait(&empty[s], (u - 1u) & 1u);
                const int p0 = (int)tile_px(i);
                const uint32_t dst = smem_u32(stages + (size_t)s * g.stage_bytes);
                mbar_expect_tx(&full[s], tx_bytes);
                if (g.Xt) {                              // tile-major copies: one contiguous block each
                    const size_t off = ((size_t)b * g.n_tiles + (size_t)(p0 / ST_PX)) * N * ST_PX;
                    bulk_load(dst, g.Xt + off, (uint32_t)N * 128u, &full[s]);
                    bulk_load(dst + g.xbytes, g.Ot + off, (uint32_t)N * 128u, &full[s]);
                } else {
                    tma_load_2d(dst, &g.mX, p0, b * N, &full[s]);
                    tma_load_2d(dst + g.xbytes, &g.mO, p0, b * N, &full[s]);
                }
                tma_load_2d(dst + 2 * g.xbytes, &g.mH, p0, b * K, &full[s]);
            }
        }
        return;
    }
    // =========================== compute warps ===========================
    const int grp = warp / ST_GWARPS, gw = warp - grp * ST_GWARPS, gt = tid - grp * ST_GTHREADS;
    float* red = red0 + grp * ST_GWARPS * 2 * K * ST_PX;
    float* hn = hn0 + grp * K * ST_PX;
    auto group_sync = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + grp), "n"(ST_GTHREADS) : "memory"); };
    // W half-step role: frame pair j = gt / 2 (frames j and j + NH), pixels 16 hf .. 16 hf + 15
    const int j = gt >> 1, hf = gt & 1;
    const int nA = j, nB = j + NH;
    const bool okA = j < NH, okB = okA && nB < N;
    float wA[K], wB[K], accA[2 * K], accB[2 * K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        wA[k] = okA ? Ws[nA * KP4 + k] : 0.f;
        wB[k] = okB ? Ws[nB * KP4 + k] : 0.f;
        accA[k] = accA[K + k] = accB[k] = accB[K + k] = 0.f;
    }
    // H half-step role: lane = pixel, frames gw, gw + 8, ...: n & 7 == gw, so the swizzled column is fixed
    const int hcol = (((lane >> 2) ^ gw) << 4) | ((lane & 3) << 2);

    for (uint32_t it = 0; it < n_my; ++it) {
        const uint32_t s = it % NS;
        mbar_wait(&full[s], (it / NS) & 1u);
        if ((int)(it & 1u) != grp) {                     // the other group's tile: observed only
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
            continue;
        }
        const unsigned char* xs = stages + (size_t)s * g.stage_bytes;
        const unsigned char* os = xs + g.xbytes;
        const float* hs = reinterpret_cast<const float*>(xs + 2 * g.xbytes);      // [K][32]
        const long long p0 = tile_px(it);
        // ---------------- H half-step ----------------
        {
            float h[K], num[K], den[K];
#pragma unroll
            for (int k = 0; k < K; ++k) { h[k] = hs[k * ST_PX + lane]; num[k] = 0.f; den[k] = 0.f; }
            const unsigned char* xr = xs + gw * 128 + hcol;
            const unsigned char* orow = os + gw * 128 + hcol;
            const float* wr = Ws + gw * KP4;
#pragma unroll 4
            for (int n = gw; n < N; n += ST_GWARPS, xr += ST_GWARPS * 128, orow += ST_GWARPS * 128, wr += ST_GWARPS * KP4) {
                const float x = *reinterpret_cast<const float*>(xr);
                const float o = *reinterpret_cast<const float*>(orow);
                float w[KP4];
#pragma unroll
                for (int k4 = 0; k4 < KP4; k4 += 4) {
                    const float4 v = *reinterpret_cast<const float4*>(wr + k4);
                    w[k4] = v.x; w[k4 + 1] = v.y; w[k4 + 2] = v.z; w[k4 + 3] = v.w;
                }
                float sv = 0.f;
#pragma unroll
                for (int k = 0; k < K; ++k) sv = fmaf(w[k], h[k], sv);
                const bool live = o > 0.f;
                const float q = live ? o * x : 0.f, r = live ? o * sv : 0.f;
#pragma unroll
                for (int k = 0; k < K; ++k) { num[k] = fmaf(w[k], q, num[k]); den[k] = fmaf(w[k], r, den[k]); }
            }
#pragma unroll
            for (int k = 0; k < K; ++k) {
                red[(gw * 2 * K + k) * ST_PX + lane] = num[k];
                red[(gw * 2 * K + K + k) * ST_PX + lane] = den[k];
            }
        }
        group_sync();
        if (gt < K * ST_PX) {                            // thread = (component k, pixel): the group's warps in order
            const int k = gt >> 5;
            float num = 0.f, den = 0.f;
#pragma unroll
            for (int w = 0; w < ST_GWARPS; ++w) {
                num += red[(w * 2 * K + k) * ST_PX + lane];
                den += red[(w * 2 * K + K + k) * ST_PX + lane];
            }
            const float hv = (hs[k * ST_PX + lane] * num) / fmaxf(den, NMF_EPS);
            hn[k * ST_PX + lane] = hv;
            if (p0 + lane < g.P) Hg[(size_t)k * g.P + p0 + lane] = hv;
        }
        group_sync();
        // ---------------- W half-step: thread = (frames nA, nB; pixels 16 hf .. 16 hf + 15) ----------------
        if (okA) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int c = 4 * hf + i;                // 16-byte chunk = 4 pixels
                float4 h4[K];
#pragma unroll
                for (int k = 0; k < K; ++k) h4[k] = *reinterpret_cast<const float4*>(hn + k * ST_PX + 4 * c);
                auto frame = [&](int n, const float (&w)[K], float (&acc)[2 * K]) {
                    const int a = n * 128 + ((c ^ (n & 7)) << 4);
                    const float4 x = *reinterpret_cast<const float4*>(xs + a);
                    const float4 o = *reinterpret_cast<const float4*>(os + a);
                    float4 sv = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        sv.x = fmaf(w[k], h4[k].x, sv.x); sv.y = fmaf(w[k], h4[k].y, sv.y);
                        sv.z = fmaf(w[k], h4[k].z, sv.z); sv.w = fmaf(w[k], h4[k].w, sv.w);
                    }
                    float4 q, r;
                    q.x = o.x > 0.f ? o.x * x.x : 0.f; r.x = o.x > 0.f ? o.x * sv.x : 0.f;
                    q.y = o.y > 0.f ? o.y * x.y : 0.f; r.y = o.y > 0.f ? o.y * sv.y : 0.f;
                    q.z = o.z > 0.f ? o.z * x.z : 0.f; r.z = o.z > 0.f ? o.z * sv.z : 0.f;
                    q.w = o.w > 0.f ? o.w * x.w : 0.f; r.w = o.w > 0.f ? o.w * sv.w : 0.f;
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        acc[k] = fmaf(q.x, h4[k].x, fmaf(q.y, h4[k].y, fmaf(q.z, h4[k].z, fmaf(q.w, h4[k].w, acc[k]))));
                        acc[K + k] = fmaf(r.x, h4[k].x, fmaf(r.y, h4[k].y, fmaf(r.z, h4[k].z, fmaf(r.w, h4[k].w, acc[K + k]))));
                    }
                };
                frame(nA, wA, accA);
                if (okB) frame(nB, wB, accB);
            }
        }
        group_sync();                                    // the group is done with the stage (and with hn, red)
        if (lane == 0) mbar_arrive(&empty[s]);
    }
    // the two threads of a frame pair (adjacent lanes) add up; lane hf == 0 writes the group's slab (part 2 cta + group)
    float* slab = g.slab + (((size_t)b * gridDim.x + blockIdx.x) * ST_GROUPS + grp) * 2 * (size_t)N * K;
#pragma unroll
    for (int k = 0; k < 2 * K; ++k) {
        float a = accA[k], c = accB[k];
        a += __shfl_xor_sync(0xffffffffu, a, 1); c += __shfl_xor_sync(0xffffffffu, c, 1);
        if (hf == 0) {
            const int half = k / K, kk = k - half * K;
            if (okA) slab[((size_t)half * N + nA) * K + kk] = a;
            if (okB) slab[((size_t)half * N + nB) * K + kk] = c;
        }
    }
}

// fixed-order fp64 reduction of the slabs [B][parts][2][N][K] + W <- W o A / max(B, eps)      (a8)
// 256 threads = 32 part lanes x 8 elements: lane q sums parts q, q + 32, ... in order, the 32 partial sums are then
// added in lane order -- a fixed association, so the result is bitwise reproducible.
constexpr int SU_E = 8, SU_Q = 32;
__global__ void __launch_bounds__(SU_E * SU_Q)
k_w_update_stream(const float* __restrict__ slab, float* __restrict__ W, int NK, int parts) {
    __shared__ double sa[SU_Q][SU_E], sd[SU_Q][SU_E];
    const int b = blockIdx.y;
    const int e = threadIdx.x % SU_E, q = threadIdx.x / SU_E;
    const int i = blockIdx.x * SU_E + e;
    const bool ok = i < NK;
    const size_t stride = (size_t)2 * NK;
    const float* s = slab + (size_t)b * parts * stride + (ok ? i : 0);
    double a = 0.0, d = 0.0;
    if (ok) {
#pragma unroll 5
        for (int part = q; part < parts; part += SU_Q) {
            a += (double)s[(size_t)part * stride];
            d += (double)s[(size_t)part * stride + NK];
        }
    }
    sa[q][e] = a; sd[q][e] = d;
    __syncthreads();
    if (q == 0 && ok) {
#pragma unroll
        for (int r = 1; r < SU_Q; ++r) { a += sa[r][e]; d += sd[r][e]; }
        float* w = W + (size_t)b * NK + i;
        *w = (*w * (float)a) / fmaxf((float)d, NMF_EPS);
    }
}

// --------------------------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------------------------
inline int xbytes_of(int N) { return (N * 128 + 1023) / 1024 * 1024; }
inline int stage_bytes_of(int N, int K) { return (2 * xbytes_of(N) + K * 128 + 1023) / 1024 * 1024; }
inline size_t fixed_bytes_of(int N, int K) {
    const int KP4 = (K + 3) / 4 * 4;
    return sizeof(float) * ((size_t)N * KP4 + (size_t)ST_CWARPS * 2 * K * ST_PX + (size_t)ST_GROUPS * K * ST_PX) + 16 * ST_MAX_STAGES + 16;
}
inline int stages_of(int N, int K) {
    long long ns = ((long long)ST_SMEM_MAX - (long long)fixed_bytes_of(N, K)) / stage_bytes_of(N, K);
    return ns > ST_MAX_STAGES ? ST_MAX_STAGES : ns < 0 ? 0 : (int)ns;
}
inline int ctas_of(const nmf_plan* p, int batch) {
    const long long n_tiles = ((p->P + ST_PX - 1) / ST_PX + 1) / 2;      // pairs of tiles
    long long avail = p->num_sms / batch;
    if (avail < 1) avail = 1;
    if (avail > n_tiles) avail = n_tiles;
    const long long per = (n_tiles + avail - 1) / avail;      // every CTA gets `per` or `per - 1` pairs
    return (int)((n_tiles + per - 1) / per);
}

// workspace: slabs [batch][ctas][groups][2][N][K], then the tile-major copies of X and Omega (each batch x n_tiles x N x 32 floats)
inline size_t slab_bytes_of(const nmf_plan* p) {
    const size_t one = (size_t)ctas_of(p, 1) * ST_GROUPS * 2 * p->N * p->K * sizeof(float);
    const size_t all = (size_t)p->batch * ctas_of(p, p->batch) * ST_GROUPS * 2 * p->N * p->K * sizeof(float);
    return nmf_align_up(one > all ? one : all, 1024);
}
inline size_t tiled_bytes_of(const nmf_plan* p, int batch) {
    return (size_t)batch * ((p->P + ST_PX - 1) / ST_PX) * p->N * ST_PX * sizeof(float);
}

template <int K>
cudaError_t launch_stream(const StreamArgs& a, dim3 grid, size_t smem, cudaStream_t st, int device) {
    static bool done[NMF_MAX_DEVICES] = {};                   // the opt-in shared-memory size is a per-device attribute
    if (!(device >= 0 && device < NMF_MAX_DEVICES && done[device])) {
        cudaError_t e = cudaFuncSetAttribute(k_stream<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ST_SMEM_MAX);
        if (e != cudaSuccess) return e;
        if (device >= 0 && device < NMF_MAX_DEVICES) done[device] = true;
    }
    k_stream<K><<<grid, ST_THREADS, smem, st>>>(a);
    return cudaSuccess;
}

}  // namespace

void nmf_stream_configure(nmf_plan* p) {
    p->st_ok = false;
    if (p->K > ST_MAXK || p->N > 256) return;
    if (p->P + ST_PX >= (1LL << 31) || (long long)p->batch * p->N >= (1LL << 31)) return;   // TMA coordinates are int32
    if (stages_of(p->N, p->K) < 2) return;
    p->st_ok = true;
}

bool nmf_stream_available(const nmf_plan* p) { return p->st_ok; }

size_t nmf_stream_workspace(const nmf_plan* p) {
    if (!p->st_ok) return 0;
    return slab_bytes_of(p) + 2 * tiled_bytes_of(p, p->batch);
}

int nmf_stream_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters, int batch) {
    if (!p->st_ok) return NMF_ERR_UNSUPPORTED;
    const int N = p->N, K = p->K;
    StreamArgs a{};
    a.W = W; a.H = H; a.slab = reinterpret_cast<float*>(p->ws);
    a.N = N; a.P = p->P; a.n_tiles = (p->P + ST_PX - 1) / ST_PX;
    a.NS = stages_of(N, K); a.xbytes = xbytes_of(N); a.stage_bytes = stage_bytes_of(N, K);
    if (!(make_map(&a.mX, X, (long long)batch * N, p->P, N, ST_PX, 128) && make_map(&a.mO, Om, (long long)batch * N, p->P, N, ST_PX, 128) &&
          make_map(&a.mH, H, (long long)batch * K, p->P, K, ST_PX, 0))) {
        if (!p->sticky) { p->sticky = NMF_ERR_CUDA; p->cuda_msg = "cuTensorMapEncodeTiled failed"; }
        return NMF_ERR_CUDA;
    }
    const int ctas = ctas_of(p, batch);
    const size_t smem = (size_t)a.NS * a.stage_bytes + fixed_bytes_of(N, K);
    const int nk = N * K;
    // from tiled_min_iters(K) iterations per call X and Omega are first copied tile-major (k_tile_major says why)
    const bool tiled = iters >= tiled_min_iters(K);
    if (tiled) {
        float* xt = reinterpret_cast<float*>(static_cast<char*>(p->ws) + slab_bytes_of(p));
        float* ot = xt + tiled_bytes_of(p, batch) / sizeof(float);
        const unsigned gx = (unsigned)((a.n_tiles * 8 + 255) / 256);
        k_tile_major<<<dim3(gx, N, 2 * batch), 256, 0, p->stream>>>(X, Om, xt, ot, N, p->P, a.n_tiles);
        p->launches++;
        NMF_CUDA_TRY(p, cudaGetLastError());
        a.Xt = xt; a.Ot = ot;
    }
    int rc = nmf_run_iterations(p, tiled ? 51 : 50, X, Om, W, H, nullptr, N, batch, iters, [&]() -> int {
        const dim3 grid(ctas, batch);
        cudaError_t e = K == 1 ? launch_stream<1>(a, grid, smem, p->stream, p->device) : K == 2 ? launch_stream<2>(a, grid, smem, p->stream, p->device) :
                        K == 3 ? launch_stream<3>(a, grid, smem, p->stream, p->device) : K == 4 ? launch_stream<4>(a, grid, smem, p->stream, p->device) :
                        K == 5 ? launch_stream<5>(a, grid, smem, p->stream, p->device) : K == 6 ? launch_stream<6>(a, grid, smem, p->stream, p->device) :
                        K == 7 ? launch_stream<7>(a, grid, smem, p->stream, p->device) : launch_stream<8>(a, grid, smem, p->stream, p->device);
        NMF_CUDA_TRY(p, e);
        k_w_update_stream<<<dim3((nk + SU_E - 1) / SU_E, batch), SU_E * SU_Q, 0, p->stream>>>(a.slab, W, nk, ctas * ST_GROUPS);
        p->launches += 2;
        return NMF_OK;
    });
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

// nmf_select.cu -- closest-frame reference selection.
//
//   D[m,n] = sum over the pixels valid in both frames (omega_t[m,p] > 0 and Omega[n,p] > 0) of (T[m,p] - X[n,p])^2
//   idx[m,:] = the n_sel references with the smallest D[m,:], ties by the lower index, ascending (G19, G20).
//
// k_ref_dist: a CTA owns a pixel range and a block of 32 targets x 128 references; a thread owns 4 targets x 4
// references (16 fp32 accumulators).  Tiles of 32 pixels are staged in shared memory with the masks folded into the
// values (a masked entry is stored as NaN, so T or X may hold anything there): per pair and pixel the update is
// d = t - x; acc += max(d * d, 0)  -- max(NaN, 0) = 0 skips the pair, four ALU operations, no mask loads.  The
// direct form is used because the expanded one (t^2 - 2tx + x^2 as three matrix products) cancels catastrophically
// in fp32 when target and reference are close, which is exactly the case of interest.
// Per-CTA partial sums go to the workspace and are reduced in a fixed order in fp64 (k_ref_reduce), so the
// distances, and with them the selection, are bitwise reproducible.  k_ref_select ranks each target's N <= 256
// distances with one thread per reference.
#include "nmf_common.cuh"
#include <math.h>

namespace {

constexpr int SD_THREADS = 256;
constexpr int SD_MB = 32;        // targets per CTA
constexpr int SD_NB = 128;       // references per CTA
constexpr int SD_TP = 32;        // pixels per staged tile
constexpr int SD_LD = SD_TP + 4; // shared-memory row stride (floats): conflict-free 128-bit reads

__global__ void __launch_bounds__(SD_THREADS)
k_ref_dist(const float* __restrict__ T, const float* __restrict__ ot, const float* __restrict__ X,
           const float* __restrict__ Om, float* __restrict__ part, int M, int N, long long P, int m0,
           long long px_per_cta) {
    __shared__ __align__(16) float ts[SD_MB][SD_LD];
    __shared__ __align__(16) float xs[SD_NB][SD_LD];
    const int n0 = blockIdx.y * SD_NB;
    const long long p_lo = (long long)blockIdx.x * px_per_cta;
    const long long p_hi = p_lo + px_per_cta < P ? p_lo + px_per_cta : P;
    const int mi = threadIdx.x >> 5, ni = threadIdx.x & 31;     // targets 4 mi + i, references ni + 32 j
    const float qnan = __int_as_float(0x7fc00000);
    float acc[4][4], tot[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) tot[i][j] = 0.f;

    // staging: (SD_MB + SD_NB) rows x 8 float4 per tile = SD_LOADS float4 per thread and array, prefetched one tile
    // ahead into registers (values and masks are loaded unconditionally and independently, then selected)
    constexpr int SD_LOADS = (SD_MB + SD_NB) * (SD_TP / 4) / SD_THREADS;     // 5
    float4 rv[SD_LOADS], rm[SD_LOADS];
    auto fetch = [&](long long pt) {
#pragma unroll
        for (int u = 0; u < SD_LOADS; ++u) {
            const int i = threadIdx.x + u * SD_THREADS;
            const int r = i >> 3, c4 = i & 7;
            const long long p = pt + 4 * c4;
            const bool is_t = r < SD_MB;
            const int row = is_t ? m0 + r : n0 + r - SD_MB;
            const bool ok = p < p_hi && (is_t ? row < M : row < N);          // P % 4 == 0: all four or none
            const float* val = is_t ? T : X;
            const float* msk = is_t ? ot : Om;
            rv[u] = make_float4(qnan, qnan, qnan, qnan);
            rm[u] = make_float4(1.f, 1.f, 1.f, 1.f);
            if (ok) {
                const size_t g = (size_t)row * P + p;
                rv[u] = __ldg(reinterpret_cast<const float4*>(val + g));
                if (msk) rm[u] = __ldg(reinterpret_cast<const float4*>(msk + g));
            }
        }
    };
    auto stash = [&]() {                                    // masked entries become NaN
#pragma unroll
        for (int u = 0; u < SD_LOADS; ++u) {
            const int i = threadIdx.x + u * SD_THREADS;
            const int r = i >> 3, c4 = i & 7;
            float4 v;
            v.x = rm[u].x > 0.f ? rv[u].x : qnan; v.y = rm[u].y > 0.f ? rv[u].y : qnan;
            v.z = rm[u].z > 0.f ? rv[u].z : qnan; v.w = rm[u].w > 0.f ? rv[u].w : qnan;
            float* dst = r < SD_MB ? &ts[r][4 * c4] : &xs[r - SD_MB][4 * c4];
            *reinterpret_cast<float4*>(dst) = v;
        }
    };
    if (p_lo < p_hi) fetch(p_lo);
    for (long long pt = p_lo; pt < p_hi; pt += SD_TP) {
        stash();
        __syncthreads();
        if (pt + SD_TP < p_hi) fetch(pt + SD_TP);           // in flight during the compute of this tile
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
#pragma unroll 2
        for (int c = 0; c < SD_TP; c += 4) {
            float4 tv[4], xv[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) tv[i] = *reinterpret_cast<const float4*>(&ts[4 * mi + i][c]);
#pragma unroll
            for (int j = 0; j < 4; ++j) xv[j] = *reinterpret_cast<const float4*>(&xs[ni + 32 * j][c]);
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float d;
                    d = tv[i].x - xv[j].x; acc[i][j] += fmaxf(d * d, 0.f);
                    d = tv[i].y - xv[j].y; acc[i][j] += fmaxf(d * d, 0.f);
                    d = tv[i].z - xv[j].z; acc[i][j] += fmaxf(d * d, 0.f);
                    d = tv[i].w - xv[j].w; acc[i][j] += fmaxf(d * d, 0.f);
                }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)                          // two-level sum: short fp32 chains
#pragma unroll
            for (int j = 0; j < 4; ++j) tot[i][j] += acc[i][j];
        __syncthreads();
    }
    // partial slab of this pixel range: [part][SD_MB][N]
    float* out = part + (size_t)blockIdx.x * SD_MB * N;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = n0 + ni + 32 * j;
            if (n < N) out[(size_t)(4 * mi + i) * N + n] = tot[i][j];
        }
}

// D[m0 + r, n] = sum over the parts in index order, fp64
__global__ void k_ref_reduce(const float* __restrict__ part, float* __restrict__ D, int M, int N, int m0, int parts) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= SD_MB * N) return;
    const int r = i / N, n = i - r * N;
    if (m0 + r >= M) return;
    double s = 0.0;
    for (int q = 0; q < parts; ++q) s += (double)part[(size_t)q * SD_MB * N + i];
    D[(size_t)(m0 + r) * N + n] = (float)s;
}

// one CTA per target, one thread per reference: rank under the order (distance, index)
__global__ void k_ref_select(const float* __restrict__ D, int N, int n_sel, int* __restrict__ idx) {
    __shared__ float d[NMF_MAX_N];
    const int m = blockIdx.x, n = threadIdx.x;
    if (n < N) d[n] = D[(size_t)m * N + n];
    __syncthreads();
    if (n >= N) return;
    const float dn = d[n];
    int rank = 0;
    for (int j = 0; j < N; ++j) rank += (d[j] < dn || (d[j] == dn && j < n)) ? 1 : 0;
    if (rank < n_sel) idx[(size_t)m * n_sel + rank] = n;
}

int ref_parts(const nmf_plan* p) {
    const int nblk = (p->N + SD_NB - 1) / SD_NB;
    int parts = 2 * p->num_sms / nblk;
    const long long tiles = (p->P + SD_TP - 1) / SD_TP;
    if (parts > tiles) parts = (int)tiles;
    return parts < 1 ? 1 : parts;
}

}  // namespace

size_t nmf_select_workspace(const nmf_plan* p) {
    return (size_t)ref_parts(p) * SD_MB * p->N * sizeof(float);
}

int nmf_select_distance(nmf_plan* p, const float* T, const float* ot, const float* X, const float* Om, int M, float* D) {
    const int parts = ref_parts(p);
    long long per = ((p->P + parts - 1) / parts + SD_TP - 1) / SD_TP * SD_TP;      // whole tiles per CTA
    float* part = reinterpret_cast<float*>(p->ws);
    const dim3 grid(parts, (p->N + SD_NB - 1) / SD_NB);
    for (int m0 = 0; m0 < M; m0 += SD_MB) {
        k_ref_dist<<<grid, SD_THREADS, 0, p->stream>>>(T, ot, X, Om, part, M, p->N, p->P, m0, per);
        k_ref_reduce<<<(SD_MB * p->N + 255) / 256, 256, 0, p->stream>>>(part, D, M, p->N, m0, parts);
        p->launches += 2;
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

int nmf_select_topn(nmf_plan* p, const float* D, int M, int n_sel, int* idx) {
    k_ref_select<<<M, NMF_MAX_N, 0, p->stream>>>(D, p->N, n_sel, idx);
    p->launches++;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

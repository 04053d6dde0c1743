// nmf_tcsplit.cu -- the two half-steps of Eq. 3 as two persistent tcgen05 kernels, K <= 128.
//
// The fused kernel of nmf_tcfit.cu keeps Num/Den, S, the piece buffers AND the persistent W-phase accumulators
// of two 128-frame M tiles in the 512 TMEM columns, and W and the H tile pieces in shared memory: that fills both
// memories at K = 64 and leaves no column to feed the H-phase S stage from TMEM.  Here the iteration is split:
//
//   k_tc_h<KS>  H half-step (a1-a5).  TMEM lane = pixel.  No W-phase accumulators, so the BF16 pieces of the H
//               tile live in TMEM (all three when they fit, else pieces 1 and 2 with piece 3 in shared memory) and
//               the S stage reads its A operand from TMEM: it runs at the tensor rate and stops competing for the
//               shared-memory port.  Num/Den take 2 KP columns, so KP = 16 KS goes up to 128 components.
//               W (3 BF16 pieces, [frames][comps]) is resident in shared memory as in the fused kernel.
//   k_tc_w<KS>  W half-step (a6-a7) with the new H.  TMEM lane = frame.  One 128-frame M tile per CTA
//               (blockIdx.z), so a CTA keeps 2 KP accumulator columns (<= 256) and its M tile's rows of W stay in
//               TMEM for the whole launch (pieces 1, 2; piece 3 in shared memory when KP > 80).  X and Omega rows
//               are read only by the CTAs of their M tile.  Also the projection kernel (a9) with X = targets,
//               Omega = omega, W = coef.
//   k_w_update_split   fixed-order fp64 reduction of the per-CTA slabs + W <- W o A / max(B, eps)  (a8)
//
// X and Omega cross HBM twice per iteration instead of once (the fused kernel re-reads them through L2), which
// the roofline of this path accounts for: it is chosen where it is faster (K > 64 always: the fused kernel does
// not exist there; K <= 64 per measurement, see nmf_tcsplit_prefer()).
// Arithmetic, operand layouts, ring and barrier protocol are those of nmf_tcfit.cu (BF16x3 split, six piece
// products per product, FP32 accumulation in TMEM, R1 / R2 written back over S in place).
#include <cuda.h>
#include "nmf_common.cuh"
#include "nmf_tc.cuh"

namespace {
using namespace tc;

constexpr int EW_WARPS = 8;               // two groups of four (one thread per TMEM lane in each group)
constexpr int W_MMA = 8, W_TMA = 9;
constexpr int THREADS = 320;
constexpr int TILE = 128;                 // pixels per tile
constexpr int FCH = 16;                   // frames per H-step chunk (one UMMA K step)
constexpr int PCH = 16;                   // pixels per W-step chunk
constexpr int NCH2 = TILE / PCH;
constexpr int HS_SB = 16 * 128;           // [128 rows][comps] piece buffers: bytes between 8-component groups
constexpr int SLOT = 16384;               // ring slot bytes (k_tc_h)
constexpr int PSW = 32;                   // k_tc_w: pixels per ring slot = one super-chunk (two W-step chunks)
constexpr int NSW = TILE / PSW;           // k_tc_w: X / Omega slots per tile
constexpr int SLOTW = 32768;              // k_tc_w ring slot bytes: [64 comps][128 px] of H, or [128 frames][32 px] of X and of Omega
constexpr int MAX_SLOTS = 8;
constexpr size_t SMEM_MAX = 227 * 1024;

struct SplitArgs {
    CUtensorMap mH;            // H   [B*K, P]  box [32 comps][128 px] (k_tc_h) or [64 comps][128 px] (k_tc_w)
    CUtensorMap mX, mO;        // X, Om [B*rows, P]: box [16 frames][128 px] (k_tc_h) or [128 frames][32 px], 128-byte swizzle
                               // (k_tc_w: full 128-byte lines from HBM; 64-byte rows ran the kernel at a quarter of the HBM rate)
    const float* W; float* H; float* slab;
    int N, K; long long P; long long n_tiles;
    int NF;                    // frames padded to a multiple of 16
    int NC;                    // H-step chunks = NF / 16
    int KH;                    // TMA slots of the H tile (32 components each in k_tc_h, 64 in k_tc_w)
    int NS;                    // ring slots
};

enum { B_HS = 0, B_S0, B_S1, B_P0, B_P1, B_G0, B_G1, B_DONE, B_FULL, B_EMPTY = B_FULL + MAX_SLOTS, B_COUNT = B_EMPTY + MAX_SLOTS };

// piece pairs (a, b) of a product, small products first: a1b3 a3b1 a2b2 a1b2 a2b1 a1b1
__device__ constexpr int PA[6] = {0, 2, 1, 0, 1, 0}, PB[6] = {2, 0, 1, 1, 0, 0};

struct RingCtl {                          // ring slot arithmetic shared by producer and consumers
    uint32_t NS, magic;
    __device__ uint32_t slot(uint32_t seq, uint32_t& par) const {
        const uint32_t qd = __umulhi(seq, magic);      // seq / NS for seq < 2^29
        par = qd & 1u;
        return seq - qd * NS;
    }
};

// 32 components (rows of a [32][128] fp32 ring slot) of pixel / frame `t` -> three words arrays of 16 (BF16 pairs)
__device__ __forceinline__ void split_slot32(const float* sl, int t, int k_base, int K, uint32_t (&p1)[16], uint32_t (&p2)[16],
                                             uint32_t (&p3)[16]) {
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const int k0 = k_base + 2 * j;
        const float h0 = k0 < K ? sl[(2 * j) * TILE + t] : 0.f;       // pixels >= P arrive zero-filled
        const float h1 = k0 + 1 < K ? sl[(2 * j + 1) * TILE + t] : 0.f;
        split3_pair(h0, h1, p1[j], p2[j], p3[j]);
    }
}
__device__ __forceinline__ void st_piece_smem(unsigned char* base, int t, int kg, const uint32_t* w) {
    *reinterpret_cast<uint4*>(base + (t & 7) * 16 + (t >> 3) * 128 + kg * HS_SB) = make_uint4(w[0], w[1], w[2], w[3]);
}
// 32 components' worth of one piece (16 words) into TMEM columns col .. col + 15 of this thread's lane; `ncol` (16 or
// 8) columns exist (the last 32-component slot is half used when KP % 32 == 16)
__device__ __forceinline__ void st_piece_tmem(uint32_t taddr, const uint32_t (&w)[16], int ncol) {
    if (ncol >= 16) tmem_st16(taddr, w);
    else { const uint32_t h[8] = {w[0], w[1], w[2], w[3], w[4], w[5], w[6], w[7]}; tmem_st8(taddr, h); }
}

// =====================================================================================================================
// H half-step
// =====================================================================================================================
template <int KS>
__global__ void __launch_bounds__(THREADS, 1)
k_tc_h(const __grid_constant__ SplitArgs g) {
    constexpr int KP = 16 * KS;
    constexpr int NPT = (2 * KP + 3 * KP / 2 + 128 <= 512) ? 3 : 2;       // H pieces kept in TMEM
    constexpr uint32_t T_NUM = 0, T_DEN = KP, T_HT = 2 * KP;              // piece i of the H tile at T_HT + i KP / 2
    constexpr uint32_t T_Z = 2 * KP + NPT * KP / 2, T_E = T_Z + 64;       // Z[jb] at T_Z + 32 jb, E[g] at T_E + 32 g
    static_assert(T_E + 64 <= 512, "TMEM");
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K, NF = g.NF, NC = g.NC, KH = g.KH;
    const long long P = g.P;
    const int WS_SB = (NF / 8) * 128;                   // Ws: bytes between 8-component groups
    const int WS_BYTES = (KP / 8) * WS_SB;
    unsigned char* ring = smem;                         // NS slots of 16 KB
    unsigned char* ws_p = ring + (size_t)g.NS * SLOT;   // 3 pieces of W
    unsigned char* hs3_p = ws_p + 3 * WS_BYTES;         // piece 3 of the H tile (NPT == 2 only)
    uint64_t* bars = reinterpret_cast<uint64_t*>(hs3_p + (NPT == 2 ? (KP / 8) * HS_SB : 0));
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);
    const RingCtl rc{(uint32_t)g.NS, 0xffffffffu / (uint32_t)g.NS + 1u};

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    float* __restrict__ H = g.H + (size_t)b * K * P;

    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_WARPS); mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1);
        mbar_init(&bars[B_P0], 4); mbar_init(&bars[B_P1], 4); mbar_init(&bars[B_G0], 1); mbar_init(&bars[B_G1], 1);
        mbar_init(&bars[B_DONE], 1);
        for (int s = 0; s < g.NS; ++s) { mbar_init(&bars[B_FULL + s], 1); mbar_init(&bars[B_EMPTY + s], 4); }
        mbar_fence_init();
    }
    if (warp == W_MMA) tmem_alloc(tptr, 512);
    if (warp == W_TMA && lane == 0) { tma_prefetch_desc(&g.mH); tma_prefetch_desc(&g.mX); tma_prefetch_desc(&g.mO); }
    for (int i = tid; i < NF * (KP / 8); i += THREADS) {    // (frame n, component group kg): 8 values -> 3 x 16 B
        const int n = i / (KP / 8), kg = i - n * (KP / 8);
        uint32_t p1[4], p2[4], p3[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int k0 = kg * 8 + 2 * j;
            const float w0 = (n < N && k0 < K) ? W[(size_t)n * K + k0] : 0.f;
            const float w1 = (n < N && k0 + 1 < K) ? W[(size_t)n * K + k0 + 1] : 0.f;
            split3_pair(w0, w1, p1[j], p2[j], p3[j]);
        }
        const uint32_t off = (n & 7) * 16 + (n >> 3) * 128 + kg * WS_SB;
        *reinterpret_cast<uint4*>(ws_p + off) = make_uint4(p1[0], p1[1], p1[2], p1[3]);
        *reinterpret_cast<uint4*>(ws_p + WS_BYTES + off) = make_uint4(p2[0], p2[1], p2[2], p2[3]);
        *reinterpret_cast<uint4*>(ws_p + 2 * WS_BYTES + off) = make_uint4(p3[0], p3[1], p3[2], p3[3]);
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tptr;
    const uint32_t ws_s = smem_u32(ws_p), hs3_s = smem_u32(hs3_p), ring_s = smem_u32(ring);
    const uint32_t slots_per_tile = (uint32_t)(KH + NC);
    const int NSC = (NC + 1) / 2;                        // super-chunks of 32 frames (the last may hold 16)

    if (warp == W_TMA) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            uint32_t seq = 0;
            auto acquire = [&]() -> uint32_t {            // next ring slot, armed for one full slot
                uint32_t par;
                const uint32_t s = rc.slot(seq, par);
                mbar_wait(&bars[B_EMPTY + s], par ^ 1u);
                mbar_expect_tx(&bars[B_FULL + s], SLOT);
                ++seq;
                return s;
            };
            for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
                const int p0 = (int)(tile * TILE);
                for (int h = 0; h < KH; ++h) {
                    const uint32_t s = acquire();
                    tma_load_2d(ring_s + s * SLOT, &g.mH, p0, b * K + 32 * h, &bars[B_FULL + s]);
                }
                for (int c = 0; c < NC; ++c) {
                    const uint32_t s = acquire();
                    tma_load_2d(ring_s + s * SLOT, &g.mX, p0, b * N + FCH * c, &bars[B_FULL + s]);
                    tma_load_2d(ring_s + s * SLOT + FCH * TILE * 4, &g.mO, p0, b * N + FCH * c, &bars[B_FULL + s]);
                }
            }
        }
    } else if (warp == W_MMA) {
        // =========================== MMA issuer (whole warp converged; one elected lane issues) ===========================
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; tc_fence_after(); };
        constexpr uint32_t id_s32 = idesc_bf16(128, 32, 0), id_s16 = idesc_bf16(128, 16, 0), id_nd = idesc_bf16(128, KP, 1);
        uint64_t d_ws_k[3], d_ws_mn[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            d_ws_k[i] = smem_desc(ws_s + i * WS_BYTES, WS_SB, 128);
            d_ws_mn[i] = smem_desc(ws_s + i * WS_BYTES, 128, WS_SB);
        }
        const uint64_t d_hs3_k = smem_desc(hs3_s, HS_SB, 128);
        const uint32_t ws_kstep = (uint32_t)(2 * WS_SB) >> 4;
        constexpr uint32_t hs_kstep = (uint32_t)(2 * HS_SB) >> 4;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
            auto issue_S = [&](int j) {                  // S(j): [128 px] x [32 frames], K = comps -> Z[j & 1]
                if (elect_one()) {
                    const uint32_t d = tmem + T_Z + 32 * (j & 1);
                    const uint32_t boff = (uint32_t)(j * 4 * 128) >> 4;
                    const uint32_t id = (2 * j + 1 < NC) ? id_s32 : id_s16;
#pragma unroll
                    for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                        for (int ks = 0; ks < KS; ++ks) {
                            const uint64_t bd = d_ws_k[PB[pr]] + boff + ks * ws_kstep;
                            if (PA[pr] < NPT) mma16_ts(d, tmem + T_HT + PA[pr] * (KP / 2) + 8 * ks, bd, id, (pr | ks) ? 1u : 0u);
                            else mma16_ss(d, d_hs3_k + ks * hs_kstep, bd, id, (pr | ks) ? 1u : 0u);
                        }
                    mma_commit(&bars[B_S0 + (j & 1)]);
                }
                __syncwarp();
            };
            wait(B_HS);
            issue_S(0);
            if (NSC > 1) issue_S(1);
            for (int j = 0; j < NSC; ++j) {
                for (int gg = 0; gg < 2; ++gg) {
                    const int c = 2 * j + gg;
                    if (c >= NC) break;
                    wait(B_P0 + gg);
                    if (elect_one()) {
                        const uint32_t z = tmem + T_Z + 32 * (j & 1) + 16 * gg, e = tmem + T_E + 32 * gg;
                        const uint32_t a_q[3] = {e + O_Q1, e + O_Q2, e + O_Q3};
                        const uint32_t a_r[3] = {z, z + 8, e + O_R3};
                        const uint32_t boff = (uint32_t)(c * 2 * 128) >> 4;   // 16 frames = 2 row groups
#pragma unroll
                        for (int pr = 0; pr < 6; ++pr) {
                            const uint32_t acc = (c > 0 || pr > 0) ? 1u : 0u;
                            mma16_ts(tmem + T_NUM, a_q[PA[pr]], d_ws_mn[PB[pr]] + boff, id_nd, acc);
                            mma16_ts(tmem + T_DEN, a_r[PA[pr]], d_ws_mn[PB[pr]] + boff, id_nd, acc);
                        }
                        mma_commit(&bars[B_G0 + gg]);
                    }
                    __syncwarp();
                }
                if (j + 2 < NSC) issue_S(j + 2);
            }
            if (elect_one()) mma_commit(&bars[B_DONE]);
            __syncwarp();
        }
    } else if (warp < EW_WARPS) {
        // =========================== element-wise warps ===========================
        const int q = warp & 3, grp = warp >> 2;
        const int t = 32 * q + lane;                     // TMEM lane = pixel of the tile
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; };
        auto wait_full = [&](uint32_t seq) -> const unsigned char* {
            uint32_t par;
            const uint32_t s = rc.slot(seq, par);
            mbar_wait(&bars[B_FULL + s], par);
            return ring + (size_t)s * SLOT;
        };
        auto release = [&](uint32_t seq) {
            __syncwarp();
            uint32_t par;
            if (lane == 0) mbar_arrive(&bars[B_EMPTY + rc.slot(seq, par)]);
        };
        auto warp_arrive = [&](int bar) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[bar]);
        };
        uint32_t sq = 0;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, sq += slots_per_tile) {
            const long long p = tile * TILE + t;
            const bool p_ok = p < P;
            const long long pc = p_ok ? p : P - 1;

            // ---- H0: the H tile's pieces -> TMEM (A operand of S); group g takes the 32-component slots g, g + 2, ...
            // (every MMA of the previous tile is complete: this warp waited for B_DONE in its update step)
            for (int h = grp; h < KH; h += 2) {
                const float* hsl = reinterpret_cast<const float*>(wait_full(sq + h));
                uint32_t p1[16], p2[16], p3[16];
                split_slot32(hsl, t, 32 * h, K, p1, p2, p3);
                release(sq + h);
                const int ncol = KP / 2 - 16 * h;        // columns of this slot that exist (16, or 8 in a half-used last slot)
                if (ncol > 0) {
                    st_piece_tmem(lane_base + T_HT + 16 * h, p1, ncol);
                    st_piece_tmem(lane_base + T_HT + KP / 2 + 16 * h, p2, ncol);
                    if (NPT == 3) st_piece_tmem(lane_base + T_HT + KP + 16 * h, p3, ncol);
                    else {
#pragma unroll
                        for (int gq = 0; gq < 4; ++gq)
                            if (4 * h + gq < KP / 8) st_piece_smem(hs3_p, t, 4 * h + gq, &p3[4 * gq]);
                    }
                }
            }
            tmem_wait_st();
            if (NPT == 2) fence_proxy_async();
            tc_fence_before();
            warp_arrive(B_HS);

            // ---- steps: super-chunk j = chunks 2j (group 0) and 2j + 1 (group 1); thread = (pixel t, 16 frames) ----
            bool pending = false;
            for (int j = 0; j < NSC; ++j) {
                const int c = 2 * j + grp;
                const bool have = c < NC;
                float x[16], o[16];
                if (have) {
                    const float* xs = reinterpret_cast<const float*>(wait_full(sq + KH + c)) + t;
                    const int nv = N - FCH * c;          // valid frames of this chunk (>= 16: all)
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        x[i] = xs[i * TILE];
                        o[i] = i < nv ? xs[FCH * TILE + i * TILE] : 0.f;
                    }
                }
                wait(B_S0 + (j & 1));                    // both groups track every completion of the buffer's barrier
                if (have) {
                    tc_fence_after();
                    const uint32_t zcol = lane_base + T_Z + 32 * (j & 1) + 16 * grp;
                    uint32_t s[16], e[32];
                    tmem_ld16(zcol, s);
                    tmem_wait_ld();
                    ew16(x, o, s, zcol, e);
                    release(sq + KH + c);                // after the values were consumed
                    if (pending) { wait(B_G0 + grp); tc_fence_after(); }
                    tmem_st32(lane_base + T_E + 32 * grp, e);
                    tmem_wait_st();
                    tc_fence_before();
                    warp_arrive(B_P0 + grp);
                    pending = true;
                }
            }
            // ---- update: h' = h * num / max(den, eps) in place; thread = (pixel t, this group's half of the comps);
            // the old h is re-read from global memory (it was loaded by TMA a moment ago: L2) ----
            if (pending) wait(B_G0 + grp);
            wait(B_DONE);                                // Num, Den complete; every S has read the H pieces
            tc_fence_after();
            {
                constexpr int NKG = KP / 8;              // 8-component groups; group g updates NKG / 2 of them
                for (int kg = grp * (NKG / 2); kg < (grp + 1) * (NKG / 2); ++kg) {
                    float* hp = H + (size_t)(8 * kg) * P + pc;
                    float hold[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) hold[j] = (8 * kg + j < K) ? hp[(size_t)j * P] : 0.f;
                    uint32_t nm[8], dn[8];
                    tmem_ld8(lane_base + T_NUM + 8 * kg, nm);
                    tmem_ld8(lane_base + T_DEN + 8 * kg, dn);
                    tmem_wait_ld();
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const float v = __fdividef(hold[j] * __uint_as_float(nm[j]), fmaxf(__uint_as_float(dn[j]), NMF_EPS));
                        if (p_ok && 8 * kg + j < K) hp[(size_t)j * P] = v;
                    }
                }
            }
            tc_fence_before();
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == W_MMA) tmem_dealloc(tmem, 512);
}

// =====================================================================================================================
// W half-step (and projection)
// =====================================================================================================================
template <int KS>
__global__ void __launch_bounds__(THREADS, 1)
k_tc_w(const __grid_constant__ SplitArgs g) {
    constexpr int KP = 16 * KS;
    constexpr int NPT = (3 * KP / 2 + 128 <= 256) ? 3 : 2;                // W pieces of the M tile kept in TMEM
    constexpr uint32_t T_WT = 0;                                          // piece i at i KP / 2
    constexpr uint32_t T_Z = NPT * KP / 2, T_E = T_Z + 64;                // Z[jb] at T_Z + 32 jb, E[g] at T_E + 32 g
    constexpr uint32_t T_ACC = 256;                                       // A at T_ACC, B at T_ACC + KP
    static_assert(T_E + 64 <= 256 && T_ACC + 2 * KP <= 512, "TMEM");
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K, KH = g.KH;
    const long long P = g.P;
    constexpr int HS_BYTES = (KP / 8) * HS_SB;          // one BF16 piece of the H tile / of the M tile's W rows
    unsigned char* ring = smem;
    unsigned char* hs_p = ring + (size_t)g.NS * SLOTW;  // 3 pieces of the H tile, [pixel][comp]
    unsigned char* ws3_p = hs_p + 3 * HS_BYTES;         // piece 3 of this M tile's rows of W (NPT == 2 only)
    uint64_t* bars = reinterpret_cast<uint64_t*>(ws3_p + (NPT == 2 ? HS_BYTES : 0));
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);
    const RingCtl rc{(uint32_t)g.NS, 0xffffffffu / (uint32_t)g.NS + 1u};

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y, m = blockIdx.z;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    // slab of this CTA: [B][MT][ctas][2][128][KP]
    float* slab = g.slab + (((size_t)b * gridDim.z + m) * gridDim.x + blockIdx.x) * 2 * (size_t)128 * KP;

    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_WARPS); mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1);
        mbar_init(&bars[B_P0], 4); mbar_init(&bars[B_P1], 4); mbar_init(&bars[B_G0], 1); mbar_init(&bars[B_G1], 1);
        mbar_init(&bars[B_DONE], 1);
        for (int s = 0; s < g.NS; ++s) { mbar_init(&bars[B_FULL + s], 1); mbar_init(&bars[B_EMPTY + s], EW_WARPS); }
        mbar_fence_init();
    }
    if (warp == W_MMA) tmem_alloc(tptr, 512);
    if (warp == W_TMA && lane == 0) { tma_prefetch_desc(&g.mH); tma_prefetch_desc(&g.mX); tma_prefetch_desc(&g.mO); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tptr;
    const uint32_t hs_s = smem_u32(hs_p), ws3_s = smem_u32(ws3_p), ring_s = smem_u32(ring);
    const uint32_t slots_per_tile = (uint32_t)(KH + NSW);
    constexpr int NSC2 = NCH2 / 2;

    if (warp < EW_WARPS) {
        // the M tile's rows of W -> TMEM (A operand of S', fixed for the launch); lane = frame 128 m + t
        const int q = warp & 3, grp = warp >> 2, t = 32 * q + lane;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const int fr = 128 * m + t;
        for (int h = grp; 32 * h < KP; h += 2) {
            uint32_t p1[16], p2[16], p3[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int k0 = 32 * h + 2 * j;
                const float w0 = (fr < N && k0 < K) ? W[(size_t)fr * K + k0] : 0.f;
                const float w1 = (fr < N && k0 + 1 < K) ? W[(size_t)fr * K + k0 + 1] : 0.f;
                split3_pair(w0, w1, p1[j], p2[j], p3[j]);
            }
            const int ncol = KP / 2 - 16 * h;
            st_piece_tmem(lane_base + T_WT + 16 * h, p1, ncol);
            st_piece_tmem(lane_base + T_WT + KP / 2 + 16 * h, p2, ncol);
            if (NPT == 3) st_piece_tmem(lane_base + T_WT + KP + 16 * h, p3, ncol);
            else {
#pragma unroll
                for (int gq = 0; gq < 4; ++gq)
                    if (4 * h + gq < KP / 8) st_piece_smem(ws3_p, t, 4 * h + gq, &p3[4 * gq]);
            }
        }
        tmem_wait_st();
        if (NPT == 2) fence_proxy_async();
        tc_fence_before();
    }
    __syncthreads();
    tc_fence_after();

    if (warp == W_TMA) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            uint32_t seq = 0;
            auto acquire = [&]() -> uint32_t {
                uint32_t par;
                const uint32_t s = rc.slot(seq, par);
                mbar_wait(&bars[B_EMPTY + s], par ^ 1u);
                mbar_expect_tx(&bars[B_FULL + s], SLOTW);
                ++seq;
                return s;
            };
            for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
                const int p0 = (int)(tile * TILE);
                for (int h = 0; h < KH; ++h) {
                    const uint32_t s = acquire();
                    tma_load_2d(ring_s + s * SLOTW, &g.mH, p0, b * K + 64 * h, &bars[B_FULL + s]);
                }
                for (int c = 0; c < NSW; ++c) {          // the M tile's 128 rows of X and Omega, 32 px (one super-chunk) at a time
                    const uint32_t s = acquire();
                    tma_load_2d(ring_s + s * SLOTW, &g.mX, p0 + PSW * c, b * N + 128 * m, &bars[B_FULL + s]);
                    tma_load_2d(ring_s + s * SLOTW + 128 * PSW * 4, &g.mO, p0 + PSW * c, b * N + 128 * m, &bars[B_FULL + s]);
                }
            }
        }
    } else if (warp == W_MMA) {
        // =========================== MMA issuer ===========================
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; tc_fence_after(); };
        constexpr uint32_t id_s32 = idesc_bf16(128, 32, 0), id_ab = idesc_bf16(128, KP, 1);
        uint64_t d_hs_k[3], d_hs_mn[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            d_hs_k[i] = smem_desc(hs_s + i * HS_BYTES, HS_SB, 128);
            d_hs_mn[i] = smem_desc(hs_s + i * HS_BYTES, 128, HS_SB);
        }
        const uint64_t d_ws3_k = smem_desc(ws3_s, HS_SB, 128);
        constexpr uint32_t hs_kstep = (uint32_t)(2 * HS_SB) >> 4;
        bool acc_started = false;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
            auto issue_S2 = [&](int j) {                 // S'(j): [128 frames] x [32 px], K = comps -> Z[j & 1]
                if (elect_one()) {
                    const uint32_t boff = (uint32_t)(j * 4 * 128) >> 4;
                    const uint32_t d = tmem + T_Z + 32 * (j & 1);
#pragma unroll
                    for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                        for (int ks = 0; ks < KS; ++ks) {
                            const uint64_t bd = d_hs_k[PB[pr]] + boff + ks * hs_kstep;
                            if (PA[pr] < NPT) mma16_ts(d, tmem + T_WT + PA[pr] * (KP / 2) + 8 * ks, bd, id_s32, (pr | ks) ? 1u : 0u);
                            else mma16_ss(d, d_ws3_k + ks * hs_kstep, bd, id_s32, (pr | ks) ? 1u : 0u);
                        }
                    mma_commit(&bars[B_S0 + (j & 1)]);
                }
                __syncwarp();
            };
            wait(B_HS);                                  // the new H tile's pieces are in Hs
            issue_S2(0);
            issue_S2(1);
            for (int j = 0; j < NSC2; ++j) {
                for (int gg = 0; gg < 2; ++gg) {
                    const int c = 2 * j + gg;
                    wait(B_P0 + gg);
                    if (elect_one()) {
                        const uint32_t boff = (uint32_t)(c * 2 * 128) >> 4;   // 16 pixels = 2 row groups
                        const uint32_t z = tmem + T_Z + 32 * (j & 1) + 16 * gg, e = tmem + T_E + 32 * gg;
                        const uint32_t a_q[3] = {e + O_Q1, e + O_Q2, e + O_Q3};
                        const uint32_t a_r[3] = {z, z + 8, e + O_R3};
#pragma unroll
                        for (int pr = 0; pr < 6; ++pr) {
                            const uint32_t acc = (acc_started || pr > 0) ? 1u : 0u;
                            mma16_ts(tmem + T_ACC, a_q[PA[pr]], d_hs_mn[PB[pr]] + boff, id_ab, acc);
                            mma16_ts(tmem + T_ACC + KP, a_r[PA[pr]], d_hs_mn[PB[pr]] + boff, id_ab, acc);
                        }
                        mma_commit(&bars[B_G0 + gg]);
                    }
                    __syncwarp();
                    acc_started = true;
                }
                if (j + 2 < NSC2) issue_S2(j + 2);
            }
            if (elect_one()) mma_commit(&bars[B_DONE]);
            __syncwarp();
        }
    } else if (warp < EW_WARPS) {
        // =========================== element-wise warps ===========================
        const int q = warp & 3, grp = warp >> 2;
        const int t = 32 * q + lane;                     // TMEM lane = frame 128 m + t
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const int fr = 128 * m + t;
        const bool active = 128 * m + 32 * q < N;        // warp-uniform: some lane has a frame
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; };
        auto wait_full = [&](uint32_t seq) -> const unsigned char* {
            uint32_t par;
            const uint32_t s = rc.slot(seq, par);
            mbar_wait(&bars[B_FULL + s], par);
            return ring + (size_t)s * SLOTW;
        };
        auto release = [&](uint32_t seq) {
            __syncwarp();
            uint32_t par;
            if (lane == 0) mbar_arrive(&bars[B_EMPTY + rc.slot(seq, par)]);
        };
        auto warp_arrive = [&](int bar) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[bar]);
        };
        uint32_t sq = 0;
        bool first = true;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, sq += slots_per_tile) {
            // ---- H0: the (new) H tile is split into Hs[pixel][comp]; thread = pixel t; a slot holds 64 components,
            // group g takes components 64 h + 32 g .. + 31 of slot h
            if (!first) wait(B_DONE);                    // every MMA of the previous tile is complete: Hs is free
            first = false;
            for (int h = 0; h < KH; ++h) {
                const float* hsl = reinterpret_cast<const float*>(wait_full(sq + h)) + (32 * grp) * TILE;
                const int hh = 2 * h + grp;              // 32-component block
                if (32 * hh < KP) {
                    uint32_t p1[16], p2[16], p3[16];
                    split_slot32(hsl, t, 32 * hh, K, p1, p2, p3);
#pragma unroll
                    for (int gq = 0; gq < 4; ++gq)
                        if (4 * hh + gq < KP / 8) {
                            st_piece_smem(hs_p, t, 4 * hh + gq, &p1[4 * gq]);
                            st_piece_smem(hs_p + HS_BYTES, t, 4 * hh + gq, &p2[4 * gq]);
                            st_piece_smem(hs_p + 2 * HS_BYTES, t, 4 * hh + gq, &p3[4 * gq]);
                        }
                }
                release(sq + h);
            }
            fence_proxy_async();
            warp_arrive(B_HS);

            // ---- steps: super-chunk j = chunks 2j + grp; thread = (frame 128 m + t, 16 pixels) ----
            bool pending = false;
            for (int j = 0; j < NSC2; ++j) {
                const uint32_t seq = sq + KH + j;        // both groups read the super-chunk's slot: group g its pixels 16 g .. 16 g + 15
                const unsigned char* xsl = wait_full(seq);           // X rows (128 bytes each, 128-byte swizzle) at +0, Omega rows at +16 KB
                float x[16], o[16];
                if (active) {
                    if (fr < N) {
                        const int sw = t & 7;
#pragma unroll
                        for (int ch = 0; ch < 4; ++ch) {
                            const int cs = ((4 * grp + ch) ^ sw) << 4;
                            const float4 xv = *reinterpret_cast<const float4*>(xsl + t * 128 + cs);
                            const float4 ov = *reinterpret_cast<const float4*>(xsl + 128 * PSW * 4 + t * 128 + cs);
                            x[4 * ch] = xv.x; x[4 * ch + 1] = xv.y; x[4 * ch + 2] = xv.z; x[4 * ch + 3] = xv.w;
                            o[4 * ch] = ov.x; o[4 * ch + 1] = ov.y; o[4 * ch + 2] = ov.z; o[4 * ch + 3] = ov.w;
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < 16; ++i) { x[i] = 0.f; o[i] = 0.f; }
                    }
                }
                wait(B_S0 + (j & 1)); tc_fence_after();
                uint32_t e[32];
                if (active) {
                    const uint32_t zcol = lane_base + T_Z + 32 * (j & 1) + 16 * grp;
                    uint32_t s[16];
                    tmem_ld16(zcol, s);
                    tmem_wait_ld();
                    ew16(x, o, s, zcol, e);
                }
                release(seq);                            // after the values were consumed
                if (pending) { wait(B_G0 + grp); tc_fence_after(); }
                if (active) tmem_st32(lane_base + T_E + 32 * grp, e);
                tmem_wait_st();
                tc_fence_before();
                warp_arrive(B_P0 + grp);
                pending = true;
            }
            wait(B_G0 + grp);
        }
        wait(B_DONE);                                    // every MMA of the last tile is complete
        tc_fence_after();
        // ---- accumulators -> this CTA's slab [2][128][KP] (grid.x <= n_tiles: every CTA had a tile) ----
        constexpr int NCG = KP / 16;                     // 16-column groups; group g writes its share
        for (int cg = grp ? (NCG + 1) / 2 : 0; cg < (grp ? NCG : (NCG + 1) / 2); ++cg) {
            uint32_t a[16], bq[16];
            tmem_ld16(lane_base + T_ACC + 16 * cg, a);
            tmem_ld16(lane_base + T_ACC + KP + 16 * cg, bq);
            tmem_wait_ld();
            float* sa = slab + (size_t)t * KP + 16 * cg;
            float* sb = sa + (size_t)128 * KP;
#pragma unroll
            for (int j = 0; j < 16; j += 4) {
                *reinterpret_cast<uint4*>(sa + j) = make_uint4(a[j], a[j + 1], a[j + 2], a[j + 3]);
                *reinterpret_cast<uint4*>(sb + j) = make_uint4(bq[j], bq[j + 1], bq[j + 2], bq[j + 3]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == W_MMA) tmem_dealloc(tmem, 512);
}

// =====================================================================================================================
// fixed-order fp64 reduction of the slabs [B][MT][parts][2][128][KP] + W <- W o A / max(B, eps)      (a8)
// 256 threads = 32 part lanes x 8 elements: lane q sums parts q, q + 32, ... in order, the 32 partial sums are then
// added in lane order -- a fixed association, so the result is bitwise reproducible.
// =====================================================================================================================
constexpr int WU_E = 8, WU_Q = 32;
__global__ void __launch_bounds__(WU_E * WU_Q)
k_w_update_split(const float* __restrict__ slab, float* __restrict__ W, int N, int K, int KP, int parts, int MT) {
    __shared__ double sa[WU_Q][WU_E], sd[WU_Q][WU_E];
    const int b = blockIdx.y;
    const int e = threadIdx.x % WU_E, q = threadIdx.x / WU_E;
    const int i = blockIdx.x * WU_E + e;
    const bool ok = i < N * K;
    const int n = ok ? i / K : 0, k = ok ? i - n * K : 0;
    const size_t stride = (size_t)2 * 128 * KP;
    const float* s = slab + ((size_t)b * MT + (n >> 7)) * parts * stride + (size_t)(n & 127) * KP + k;
    double a = 0.0, d = 0.0;
    if (ok) {
#pragma unroll 5
        for (int part = q; part < parts; part += WU_Q) {
            a += (double)s[(size_t)part * stride];
            d += (double)s[(size_t)part * stride + (size_t)128 * KP];
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

// --------------------------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------------------------
inline int kp_of(int K) { return (K + 15) / 16 * 16; }
inline int npt_h(int KP) { return (2 * KP + 3 * KP / 2 + 128 <= 512) ? 3 : 2; }
inline int npt_w(int KP) { return (3 * KP / 2 + 128 <= 256) ? 3 : 2; }
inline size_t smem_fixed_h(int NF, int KP) {
    return (size_t)3 * KP * NF * 2 + (npt_h(KP) == 2 ? (size_t)(KP / 8) * HS_SB : 0) + B_COUNT * 8 + 16;
}
inline size_t smem_fixed_w(int KP) {
    return (size_t)(3 + (npt_w(KP) == 2 ? 1 : 0)) * (KP / 8) * HS_SB + B_COUNT * 8 + 16;
}
inline int slots_for(size_t fixed, int slot_bytes) {
    long long ns = ((long long)SMEM_MAX - (long long)fixed) / slot_bytes;
    return (int)(ns > MAX_SLOTS ? MAX_SLOTS : ns);
}

template <int KS>
cudaError_t launch_h(const SplitArgs& a, dim3 grid, size_t smem, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(k_tc_h<KS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
    if (e != cudaSuccess) return e;
    k_tc_h<KS><<<grid, THREADS, smem, st>>>(a);
    return cudaSuccess;
}
template <int KS>
cudaError_t launch_w(const SplitArgs& a, dim3 grid, size_t smem, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(k_tc_w<KS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
    if (e != cudaSuccess) return e;
    k_tc_w<KS><<<grid, THREADS, smem, st>>>(a);
    return cudaSuccess;
}
#define NMF_KS_SWITCH(fn, KS, ...)                                    \
    ((KS) == 1 ? fn<1>(__VA_ARGS__) : (KS) == 2 ? fn<2>(__VA_ARGS__) : (KS) == 3 ? fn<3>(__VA_ARGS__) : \
     (KS) == 4 ? fn<4>(__VA_ARGS__) : (KS) == 5 ? fn<5>(__VA_ARGS__) : (KS) == 6 ? fn<6>(__VA_ARGS__) : \
     (KS) == 7 ? fn<7>(__VA_ARGS__) : fn<8>(__VA_ARGS__))

// persistent CTAs for `n_tiles` tiles on `avail` SMs, evened out so that every CTA gets `per` or `per - 1` tiles
inline int even_ctas(long long n_tiles, long long avail) {
    if (avail < 1) avail = 1;
    if (avail > n_tiles) avail = n_tiles;
    const long long per = (n_tiles + avail - 1) / avail;
    return (int)((n_tiles + per - 1) / per);
}

// iters x { W half-step (+ optionally the H half-step before it) ; reduce + update }
int split_run(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int rows, int iters, int batch, bool fit) {
    const int KP = kp_of(p->K), KS = KP / 16;
    const int MT = (rows + 127) / 128;
    const long long n_tiles = (p->P + TILE - 1) / TILE;
    const long long trows = (long long)batch * rows;
    SplitArgs h{}, w{};
    h.W = w.W = W; h.H = w.H = H; w.slab = h.slab = reinterpret_cast<float*>(p->ws);
    h.N = w.N = rows; h.K = w.K = p->K; h.P = w.P = p->P; h.n_tiles = w.n_tiles = n_tiles;
    h.NF = w.NF = (rows + FCH - 1) / FCH * FCH; h.NC = w.NC = h.NF / FCH; h.KH = (p->K + 31) / 32; w.KH = (p->K + 63) / 64;
    h.NS = slots_for(smem_fixed_h(h.NF, KP), SLOT); w.NS = slots_for(smem_fixed_w(KP), SLOTW);
    bool ok = make_map(&w.mH, H, (long long)batch * p->K, p->P, 64, TILE, 0) &&
              make_map(&w.mX, X, trows, p->P, 128, PSW, 128) && make_map(&w.mO, Om, trows, p->P, 128, PSW, 128);
    if (fit) ok = ok && make_map(&h.mH, H, (long long)batch * p->K, p->P, 32, TILE, 0) &&
                  make_map(&h.mX, X, trows, p->P, FCH, TILE, 0) && make_map(&h.mO, Om, trows, p->P, FCH, TILE, 0);
    if (!ok) {
        if (!p->sticky) { p->sticky = NMF_ERR_CUDA; p->cuda_msg = "cuTensorMapEncodeTiled failed"; }
        return NMF_ERR_CUDA;
    }
    const int ctas_h = even_ctas(n_tiles, p->num_sms / batch);
    const int ctas_w = even_ctas(n_tiles, p->num_sms / (batch * MT));
    const size_t smem_h = smem_fixed_h(h.NF, KP) + (size_t)h.NS * SLOT, smem_w = smem_fixed_w(KP) + (size_t)w.NS * SLOTW;
    const int nk = rows * p->K;
    for (int it = 0; it < iters; ++it) {
        if (fit) {
            NMF_CUDA_TRY(p, NMF_KS_SWITCH(launch_h, KS, h, dim3(ctas_h, batch), smem_h, p->stream));
            p->launches++;
        }
        NMF_CUDA_TRY(p, NMF_KS_SWITCH(launch_w, KS, w, dim3(ctas_w, batch, MT), smem_w, p->stream));
        k_w_update_split<<<dim3((nk + WU_E - 1) / WU_E, batch), WU_E * WU_Q, 0, p->stream>>>(w.slab, W, rows, p->K, KP, ctas_w, MT);
        p->launches += 2;
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

}  // namespace

void nmf_tcsplit_configure(nmf_plan* p) {
    p->s_ok = false;
    if (p->K > 128 || p->N > 256) return;
    if (p->P + TILE >= (1LL << 31) || (long long)p->batch * p->N >= (1LL << 31)) return;   // TMA coordinates are int32
    const int KP = kp_of(p->K), NF = (p->N + FCH - 1) / FCH * FCH;
    if (slots_for(smem_fixed_h(NF, KP), SLOT) < 2 || slots_for(smem_fixed_w(KP), SLOTW) < 2) return;
    p->s_ok = true;
}

size_t nmf_tcsplit_workspace(const nmf_plan* p) {
    if (!p->s_ok) return 0;
    const int KP = kp_of(p->K);
    const long long n_tiles = (p->P + TILE - 1) / TILE;
    auto slabs = [&](int rows, int batch) {
        const int MT = (rows + 127) / 128;
        return (size_t)batch * MT * even_ctas(n_tiles, p->num_sms / (batch * MT)) * 2 * 128 * KP * sizeof(float);
    };
    size_t need = slabs(p->N, p->batch);
    const size_t one = slabs(p->N, 1);
    if (one > need) need = one;
    if (p->max_targets > 0) {
        const size_t pr = slabs(p->max_targets < 256 ? p->max_targets : 256, 1);
        if (pr > need) need = pr;
    }
    return need;
}

bool nmf_tcsplit_available(const nmf_plan* p) { return p->s_ok; }

int nmf_tcsplit_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters, int batch) {
    if (!p->s_ok) return NMF_ERR_UNSUPPORTED;
    return split_run(p, X, Om, W, H, p->N, iters, batch, true);
}

// Projection (a9): the W half-step kernel alone with H fixed, X = targets, Omega = omega, W = coef; 256 frames per pass.
int nmf_tcsplit_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C, int M, int iters) {
    if (!p->s_ok || !om) return NMF_ERR_UNSUPPORTED;
    for (int m0 = 0; m0 < M; m0 += 256) {
        const int rows = M - m0 < 256 ? M - m0 : 256;
        int rc = split_run(p, T + (size_t)m0 * p->P, om + (size_t)m0 * p->P, C + (size_t)m0 * p->K, const_cast<float*>(H), rows,
                           iters, 1, false);
        if (rc) return rc;
    }
    return NMF_OK;
}

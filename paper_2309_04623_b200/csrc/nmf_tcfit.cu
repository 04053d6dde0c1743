// nmf_tcfit.cu -- fused per-pixel-tile NMF iteration on the tcgen05 tensor cores.
//
// One persistent CTA (8 element-wise warps + 1 MMA-issuing warp) walks tiles of 128 pixels.  All six
// contractions of Eq. 3 run as tcgen05.mma kind::f16 on BF16 operands with FP32
// accumulation in TMEM.  Every FP32 operand x is split exactly into three BF16 pieces
// x = x1 + x2 + x3 (x1 = bf16(x), x2 = bf16(x - x1), x3 = x - x1 - x2) and a product a*b is evaluated as
// the six piece products a1b1 + a1b2 + a2b1 + a2b2 + a1b3 + a3b1 (dropped terms <= 2^-24 |ab|), so the
// arithmetic stays FP32-faithful ("BF16x3", the BF16 analogue of the 3xTF32 split; it is used instead of
// TF32 because 16-bit operands can be read both K-major and MN-major from one no-swizzle buffer, which
// lets W and H' serve two contractions each from a single shared-memory copy).
//
// Per tile (p0 .. p0+127), with W (3 pieces, [frames][comps]) resident in shared memory:
//   H phase (TMEM lane = pixel):
//     H0   the H tile is split and written to shared memory as Hs[pixel][comp]           (a1)
//     S    S^T[pixel][frame] = Hs . Ws^T, 32 frames at a time (SS MMAs, N = 32)           (a2)
//     EW   thread = (pixel, 16 frames): q = Om*X (select), r = Om*S, split -> TMEM        (a3)
//     ND   Num^T += Q^T . W, Den^T += R^T . W   (A from TMEM, B = MN-major view of Ws)    (a4)
//     UPD  h' = h * num / max(den, eps) -> global H and, split, back into Hs              (a5)
//   W phase (TMEM lane = frame, two M tiles of 128 frames), 32 pixels at a time:
//     S'   S'[frame][pixel] = Ws . Hs^T (SS MMAs, N = 32)                                 (a6)
//     EW   thread = frame: X, Om re-read (L2) through cp.async-staged swizzled sub-tiles;
//          q, r' = Om*S' split -> TMEM                                                    (a6)
//     AB   A += Q . Hs, B += R' . Hs  (A from TMEM, B = MN-major view of Hs), accumulated in TMEM
//          over all tiles of the CTA                                                      (a7)
//   After the last tile the [2][N][64] accumulators go to this CTA's slab; nmf_launch_w_update reduces
//   the slabs in fixed order and updates W (a8).
// S / S' chunks are double-buffered in TMEM; the split pieces are single-buffered, so the element-wise
// warps of chunk c+1 overlap the MMAs of chunk c except for their final piece stores.
#include "nmf_common.cuh"
#include "nmf_tc.cuh"

namespace {
using namespace tc;

constexpr int EW_THREADS = 256;            // warps 0..7
constexpr int CTA_THREADS = 288;           // + warp 8 = MMA issuer
constexpr int TILE = 128;                  // pixels per tile = UMMA M of the H phase
constexpr int CHP = 32;                    // pixels per W-phase chunk
constexpr int SUBP = 16;                   // pixels per cp.async sub-stage (64-byte rows)
constexpr int KP = 64;                     // components padded to the MN-major N of stages 2 and 4
constexpr int HS_SB = 16 * 128;            // Hs: bytes between 8-component groups (128 pixels x 16 B)
constexpr int HS_BYTES = 8 * HS_SB;        // one BF16 piece of the H tile

// TMEM columns (512 allocated)
constexpr uint32_t T_S = 0;                // H phase: S_b at 32 b; R1/R2 overwrite it in place
constexpr uint32_t T_R3 = 64;              //          R3 (+8 per k-step)
constexpr uint32_t T_Q = 80;               //          Q_j at 16 j (+8 per k-step)
constexpr uint32_t T_NUM = 128, T_DEN = 192;
constexpr uint32_t T_S2 = 0;               // W phase: S'_b[m] at 64 b + 32 m
constexpr uint32_t T_P2 = 128;             //          pieces[m] at 64 m: R'3 at +0, Q_j at 16 + 16 j
constexpr uint32_t T_ACC = 256;            // A_acc[m] at 128 m, B_acc[m] at 128 m + 64

__host__ __device__ constexpr uint32_t idesc_bf16(int M, int N, int b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
           ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma16_ss(uint32_t d, uint64_t a, uint64_t b, uint32_t id, uint32_t acc) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d), "l"(a), "l"(b), "r"(id), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma16_ts(uint32_t d, uint32_t a, uint64_t b, uint32_t id, uint32_t acc) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                 ::"r"(d), "r"(a), "l"(b), "r"(id), "r"(acc) : "memory");
}
__device__ __forceinline__ bool elect_one() {
    uint32_t p;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(p));
    return p != 0;
}
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// exact 3-way BF16 split of two FP32 values, packed (low half = first value)
__device__ __forceinline__ void split3_pair(float x0, float x1, uint32_t& p1, uint32_t& p2, uint32_t& p3) {
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(p1) : "f"(x1), "f"(x0));
    const float r0 = x0 - __uint_as_float(p1 << 16);
    const float r1 = x1 - __uint_as_float(p1 & 0xffff0000u);
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(p2) : "f"(r1), "f"(r0));
    const float s0 = r0 - __uint_as_float(p2 << 16);
    const float s1 = r1 - __uint_as_float(p2 & 0xffff0000u);
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(p3) : "f"(s1), "f"(s0));
}

__device__ __forceinline__ void cp_async16(uint32_t smem_dst, const void* gsrc, bool valid) {
    const int sz = valid ? 16 : 0;                       // src-size 0: zero-fill, nothing is read
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_dst), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N_> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N_) : "memory"); }

struct TcArgs {
    const float* X; const float* Om; const float* W; float* H; float* slab;
    int N, K; long long P; long long n_tiles;
    int NF;            // frames padded to a multiple of 32 (rows of the W pieces)
    int MT;            // 128-frame M tiles of the W phase (1 or 2)
    int KS;            // 16-component k-steps of stages 1 and 3
};

// barrier slots
enum { B_HS = 0, B_HS2, B_S0, B_S1, B_P, B_ND, B_S20, B_S21, B_P2, B_ND2, B_COUNT };

template <int NST>
__global__ void __launch_bounds__(CTA_THREADS, 1)
k_tc_iter(const TcArgs g) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K, NF = g.NF;
    const long long P = g.P;
    const int WS_SB = (NF / 8) * 128;                   // Ws: bytes between 8-component groups
    const int WS_BYTES = 8 * WS_SB;
    const int ST_ARR = N * (SUBP * 4);                  // one array (X or Om) of one sub-stage
    unsigned char* ws_p = smem;                         // 3 pieces of W
    unsigned char* hs_p = ws_p + 3 * WS_BYTES;          // 3 pieces of the H tile
    unsigned char* stg = hs_p + 3 * HS_BYTES;           // NST sub-stages of {X, Om}
    uint64_t* bars = reinterpret_cast<uint64_t*>(stg + (size_t)NST * 2 * ST_ARR);
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y;
    const float* __restrict__ X = g.X + (size_t)b * N * P;
    const float* __restrict__ Om = g.Om + (size_t)b * N * P;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    float* __restrict__ H = g.H + (size_t)b * K * P;
    float* slab = g.slab + ((size_t)b * gridDim.x + blockIdx.x) * 2 * (size_t)N * KP;

    // ---------------- setup: barriers, TMEM, W pieces ----------------
    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_THREADS); mbar_init(&bars[B_HS2], EW_THREADS);
        mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1);
        mbar_init(&bars[B_P], EW_THREADS); mbar_init(&bars[B_ND], 1);
        mbar_init(&bars[B_S20], 1); mbar_init(&bars[B_S21], 1);
        mbar_init(&bars[B_P2], EW_THREADS); mbar_init(&bars[B_ND2], 1);
        mbar_fence_init();
    }
    if (warp == 8) tmem_alloc(tptr, 512);
    for (int i = tid; i < NF * 8; i += CTA_THREADS) {   // (frame n, component group kg): 8 values -> 3 x 16 B
        const int n = i >> 3, kg = i & 7;
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
    const uint32_t ws_s = smem_u32(ws_p), hs_s = smem_u32(hs_p), stg_s = smem_u32(stg);
    const int n_chunks = NF / 32;                       // H-phase chunks of 32 frames
    constexpr int n_chunks2 = TILE / CHP;               // W-phase chunks of 32 pixels
    constexpr int n_sub = TILE / SUBP;
    constexpr int LOOK = NST - 1;

    if (warp == 8) {
        // =========================== MMA issuer ===========================
        uint32_t ph_hs = 0, ph_hs2 = 0, ph_p = 0, ph_p2 = 0;
        uint32_t acc_started = 0;
        const uint32_t id_s = idesc_bf16(128, 32, 0), id_nd = idesc_bf16(128, 64, 1);
        // piece pairs (a, b), small products first: a1b3 a3b1 a2b2 a1b2 a2b1 a1b1
        const int pa[6] = {0, 2, 1, 0, 1, 0}, pb[6] = {2, 0, 1, 1, 0, 0};
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
            // ---- H phase ----
            mbar_wait(&bars[B_HS], ph_hs); ph_hs ^= 1;
            tc_fence_after();
            for (int c = -1; c < n_chunks; ++c) {
                if (c + 1 < n_chunks) {                  // S(c+1): [128 px] x [32 frames], K = comps
                    if (elect_one()) {
                        const int cc = c + 1;
                        const uint32_t d = tmem + T_S + 32 * (cc & 1);
                        uint32_t acc = 0;
#pragma unroll
                        for (int pr = 0; pr < 6; ++pr)
                            for (int ks = 0; ks < g.KS; ++ks) {
                                const uint64_t ad = smem_desc(hs_s + pa[pr] * HS_BYTES + ks * 2 * HS_SB, HS_SB, 128);
                                const uint64_t bd = smem_desc(ws_s + pb[pr] * WS_BYTES + cc * 4 * 128 + ks * 2 * WS_SB, WS_SB, 128);
                                mma16_ss(d, ad, bd, id_s, acc);
                                acc = 1;
                            }
                        mma_commit(&bars[B_S0 + (cc & 1)]);
                    }
                    __syncwarp();
                }
                if (c >= 0) {                            // ND(c): Num^T, Den^T += pieces(c) . W
                    mbar_wait(&bars[B_P], ph_p); ph_p ^= 1;
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t sb = tmem + T_S + 32 * (c & 1);
#pragma unroll
                        for (int ks = 0; ks < 2; ++ks) {
                            const uint32_t a_q[3] = {tmem + T_Q + 8 * ks, tmem + T_Q + 16 + 8 * ks, tmem + T_Q + 32 + 8 * ks};
                            const uint32_t a_r[3] = {sb + 16 * ks, sb + 16 * ks + 8, tmem + T_R3 + 8 * ks};
                            const uint32_t frow = (uint32_t)(c * 4 + ks * 2) * 128;   // 16 frames = 2 row groups
#pragma unroll
                            for (int pr = 0; pr < 6; ++pr) {
                                const uint64_t bd = smem_desc(ws_s + pb[pr] * WS_BYTES + frow, 128, WS_SB);
                                const uint32_t acc = (c > 0 || ks > 0 || pr > 0) ? 1u : 0u;
                                mma16_ts(tmem + T_NUM, a_q[pa[pr]], bd, id_nd, acc);
                                mma16_ts(tmem + T_DEN, a_r[pa[pr]], bd, id_nd, acc);
                            }
                        }
                        mma_commit(&bars[B_ND]);
                    }
                    __syncwarp();
                }
            }
            // ---- W phase ----
            mbar_wait(&bars[B_HS2], ph_hs2); ph_hs2 ^= 1;
            tc_fence_after();
            for (int c = -1; c < n_chunks2; ++c) {
                if (c + 1 < n_chunks2) {                 // S'(c+1)[m]: [128 frames] x [32 px], K = comps
                    if (elect_one()) {
                        const int cc = c + 1;
                        for (int m = 0; m < g.MT; ++m) {
                            const uint32_t d = tmem + T_S2 + 64 * (cc & 1) + 32 * m;
                            uint32_t acc = 0;
#pragma unroll
                            for (int pr = 0; pr < 6; ++pr)
                                for (int ks = 0; ks < g.KS; ++ks) {
                                    const uint64_t ad = smem_desc(ws_s + pa[pr] * WS_BYTES + m * 16 * 128 + ks * 2 * WS_SB, WS_SB, 128);
                                    const uint64_t bd = smem_desc(hs_s + pb[pr] * HS_BYTES + cc * 4 * 128 + ks * 2 * HS_SB, HS_SB, 128);
                                    mma16_ss(d, ad, bd, id_s, acc);
                                    acc = 1;
                                }
                        }
                        mma_commit(&bars[B_S20 + (cc & 1)]);
                    }
                    __syncwarp();
                }
                if (c >= 0) {                            // AB(c): A_acc += Q . Hs, B_acc += R' . Hs
                    mbar_wait(&bars[B_P2], ph_p2); ph_p2 ^= 1;
                    tc_fence_after();
                    if (elect_one()) {
                        for (int m = 0; m < g.MT; ++m) {
                            const uint32_t sb = tmem + T_S2 + 64 * (c & 1) + 32 * m;
                            const uint32_t pb2 = tmem + T_P2 + 64 * m;
#pragma unroll
                            for (int ks = 0; ks < 2; ++ks) {
                                const uint32_t a_q[3] = {pb2 + 16 + 8 * ks, pb2 + 32 + 8 * ks, pb2 + 48 + 8 * ks};
                                const uint32_t a_r[3] = {sb + 16 * ks, sb + 16 * ks + 8, pb2 + 8 * ks};
                                const uint32_t prow = (uint32_t)(c * 4 + ks * 2) * 128;   // 16 pixels = 2 row groups
#pragma unroll
                                for (int pr = 0; pr < 6; ++pr) {
                                    const uint64_t bd = smem_desc(hs_s + pb[pr] * HS_BYTES + prow, 128, HS_SB);
                                    const uint32_t acc = (acc_started || ks > 0 || pr > 0) ? 1u : 0u;
                                    mma16_ts(tmem + T_ACC + 128 * m, a_q[pa[pr]], bd, id_nd, acc);
                                    mma16_ts(tmem + T_ACC + 128 * m + 64, a_r[pa[pr]], bd, id_nd, acc);
                                }
                            }
                        }
                        mma_commit(&bars[B_ND2]);
                    }
                    acc_started = 1;
                    __syncwarp();
                }
            }
        }
    } else {
        // =========================== element-wise warps ===========================
        const int q = warp & 3, half = warp >> 2;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        uint32_t ph_s[2] = {0, 0}, ph_nd = 0, ph_s2[2] = {0, 0}, ph_nd2 = 0;
        const int t = 32 * q + lane;                     // H phase: pixel within the tile
        const int fr = 128 * half + 32 * q + lane;       // W phase: frame
        const bool fr_ok = fr < N;
        const bool do_tm = half < g.MT;

        auto issue_sub = [&](long long p0, int s) {      // cp.async sub-stage s of the tile at p0
            if (s < n_sub) {
                const uint32_t dstb = stg_s + (uint32_t)(s % NST) * 2 * ST_ARR;
                const long long ps = p0 + (long long)s * SUBP;
                for (int i = tid; i < N * 4; i += EW_THREADS) {
                    const int row = i >> 2, ch = i & 3;
                    const long long p = ps + 4 * ch;
                    const bool ok = p < P;               // P % 4 == 0: a chunk is all in or all out
                    const size_t gi = (size_t)row * P + (ok ? p : 0);
                    const uint32_t d = dstb + row * 64 + ((ch ^ ((row >> 1) & 3)) << 4);
                    cp_async16(d, X + gi, ok);
                    cp_async16(d + ST_ARR, Om + gi, ok);
                }
            }
            cp_async_commit();
        };

        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
            const long long p0 = tile * TILE;
            const long long p = p0 + t;
            const bool p_ok = p < P;
            const long long pc = p_ok ? p : P - 1;
            named_bar_sync(1, EW_THREADS);               // every reader of the previous tile's stages is done
#pragma unroll
            for (int s = 0; s < LOOK; ++s) issue_sub(p0, s);

            // ---- H0: split the H tile into Hs[pixel][comp] ----
#pragma unroll
            for (int gq = 0; gq < 4; ++gq) {
                const int kg = 4 * half + gq;
                uint32_t p1[4], p2[4], p3[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int k0 = kg * 8 + 2 * j;
                    const float h0 = (p_ok && k0 < K) ? H[(size_t)k0 * P + pc] : 0.f;
                    const float h1 = (p_ok && k0 + 1 < K) ? H[(size_t)(k0 + 1) * P + pc] : 0.f;
                    split3_pair(h0, h1, p1[j], p2[j], p3[j]);
                }
                const uint32_t off = (t & 7) * 16 + (t >> 3) * 128 + kg * HS_SB;
                *reinterpret_cast<uint4*>(hs_p + off) = make_uint4(p1[0], p1[1], p1[2], p1[3]);
                *reinterpret_cast<uint4*>(hs_p + HS_BYTES + off) = make_uint4(p2[0], p2[1], p2[2], p2[3]);
                *reinterpret_cast<uint4*>(hs_p + 2 * HS_BYTES + off) = make_uint4(p3[0], p3[1], p3[2], p3[3]);
            }
            fence_proxy_async();
            mbar_arrive(&bars[B_HS]);

            // ---- H phase chunks: thread = (pixel t, 16 frames) ----
            for (int c = 0; c < n_chunks; ++c) {
                const int bb = c & 1;
                const int f0 = 32 * c + 16 * half;
                float x[16], o[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int n = f0 + i;
                    const bool ok = p_ok && n < N;
                    o[i] = ok ? __ldg(Om + (size_t)n * P + pc) : 0.f;
                    x[i] = ok ? __ldg(X + (size_t)n * P + pc) : 0.f;
                }
                mbar_wait(&bars[B_S0 + bb], ph_s[bb]); ph_s[bb] ^= 1;
                tc_fence_after();
                uint32_t s[16];
                const uint32_t s_addr = lane_base + T_S + 32 * bb + 16 * half;
                tmem_ld16(s_addr, s);
                tmem_wait_ld();
                uint32_t R1[8], R2[8], R3[8], Q1[8], Q2[8], Q3[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float o0 = o[2 * i], o1 = o[2 * i + 1];
                    // Omega == 0: missing datum, skipped (G5); X may be NaN/Inf there
                    const float q0 = o0 > 0.f ? o0 * x[2 * i] : 0.f;
                    const float q1 = o1 > 0.f ? o1 * x[2 * i + 1] : 0.f;
                    const float r0 = o0 > 0.f ? o0 * __uint_as_float(s[2 * i]) : 0.f;
                    const float r1 = o1 > 0.f ? o1 * __uint_as_float(s[2 * i + 1]) : 0.f;
                    split3_pair(q0, q1, Q1[i], Q2[i], Q3[i]);
                    split3_pair(r0, r1, R1[i], R2[i], R3[i]);
                }
                tmem_st8(s_addr, R1);
                tmem_st8(s_addr + 8, R2);
                if (c > 0) { mbar_wait(&bars[B_ND], ph_nd); ph_nd ^= 1; tc_fence_after(); }
                tmem_st8(lane_base + T_R3 + 8 * half, R3);
                tmem_st8(lane_base + T_Q + 8 * half, Q1);
                tmem_st8(lane_base + T_Q + 16 + 8 * half, Q2);
                tmem_st8(lane_base + T_Q + 32 + 8 * half, Q3);
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(&bars[B_P]);
            }
            mbar_wait(&bars[B_ND], ph_nd); ph_nd ^= 1;   // Num, Den complete; every stage-1 read of Hs is done
            tc_fence_after();

            // ---- UPD: h' = h * num / max(den, eps); thread = (pixel t, 32 comps) ----
#pragma unroll
            for (int gq = 0; gq < 4; ++gq) {
                const int kg = 4 * half + gq;
                uint32_t nm[8], dn[8];
                tmem_ld8(lane_base + T_NUM + 8 * kg, nm);
                tmem_ld8(lane_base + T_DEN + 8 * kg, dn);
                tmem_wait_ld();
                float hn[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int k = kg * 8 + j;
                    float v = 0.f;
                    if (p_ok && k < K) {
                        const float h = H[(size_t)k * P + pc];
                        v = (h * __uint_as_float(nm[j])) / fmaxf(__uint_as_float(dn[j]), NMF_EPS);
                        H[(size_t)k * P + pc] = v;
                    }
                    hn[j] = v;
                }
                uint32_t p1[4], p2[4], p3[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) split3_pair(hn[2 * j], hn[2 * j + 1], p1[j], p2[j], p3[j]);
                const uint32_t off = (t & 7) * 16 + (t >> 3) * 128 + kg * HS_SB;
                *reinterpret_cast<uint4*>(hs_p + off) = make_uint4(p1[0], p1[1], p1[2], p1[3]);
                *reinterpret_cast<uint4*>(hs_p + HS_BYTES + off) = make_uint4(p2[0], p2[1], p2[2], p2[3]);
                *reinterpret_cast<uint4*>(hs_p + 2 * HS_BYTES + off) = make_uint4(p3[0], p3[1], p3[2], p3[3]);
            }
            fence_proxy_async();
            tc_fence_before();
            mbar_arrive(&bars[B_HS2]);

            // ---- W phase chunks: thread = frame, 2 x 16 pixels per chunk ----
            for (int c = 0; c < n_chunks2; ++c) {
                const int bb = c & 1;
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    const int s_idx = 2 * c + hh;
                    cp_async_wait<LOOK - 1>();
                    named_bar_sync(1, EW_THREADS);
                    issue_sub(p0, s_idx + LOOK);
                    if (hh == 0) { mbar_wait(&bars[B_S20 + bb], ph_s2[bb]); ph_s2[bb] ^= 1; tc_fence_after(); }
                    uint32_t R1[8], R2[8], R3[8], Q1[8], Q2[8], Q3[8];
                    const uint32_t s_addr = lane_base + T_S2 + 64 * bb + 32 * half + 16 * hh;
                    if (do_tm) {
                        uint32_t s[16];
                        tmem_ld16(s_addr, s);
                        float x[16], o[16];
                        if (fr_ok) {
                            const unsigned char* xr = stg + (size_t)(s_idx % NST) * 2 * ST_ARR + fr * 64;
                            const int sw = (fr >> 1) & 3;
#pragma unroll
                            for (int ch = 0; ch < 4; ++ch) {
                                const float4 xv = *reinterpret_cast<const float4*>(xr + ((ch ^ sw) << 4));
                                const float4 ov = *reinterpret_cast<const float4*>(xr + ST_ARR + ((ch ^ sw) << 4));
                                x[4 * ch] = xv.x; x[4 * ch + 1] = xv.y; x[4 * ch + 2] = xv.z; x[4 * ch + 3] = xv.w;
                                o[4 * ch] = ov.x; o[4 * ch + 1] = ov.y; o[4 * ch + 2] = ov.z; o[4 * ch + 3] = ov.w;
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < 16; ++i) { x[i] = 0.f; o[i] = 0.f; }
                        }
                        tmem_wait_ld();
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            const float o0 = o[2 * i], o1 = o[2 * i + 1];
                            const float q0 = o0 > 0.f ? o0 * x[2 * i] : 0.f;
                            const float q1 = o1 > 0.f ? o1 * x[2 * i + 1] : 0.f;
                            const float r0 = o0 > 0.f ? o0 * __uint_as_float(s[2 * i]) : 0.f;
                            const float r1 = o1 > 0.f ? o1 * __uint_as_float(s[2 * i + 1]) : 0.f;
                            split3_pair(q0, q1, Q1[i], Q2[i], Q3[i]);
                            split3_pair(r0, r1, R1[i], R2[i], R3[i]);
                        }
                        tmem_st8(s_addr, R1);
                        tmem_st8(s_addr + 8, R2);
                    }
                    if (hh == 0 && c > 0) { mbar_wait(&bars[B_ND2], ph_nd2); ph_nd2 ^= 1; tc_fence_after(); }
                    if (do_tm) {
                        const uint32_t pbase = lane_base + T_P2 + 64 * half + 8 * hh;
                        tmem_st8(pbase, R3);
                        tmem_st8(pbase + 16, Q1);
                        tmem_st8(pbase + 32, Q2);
                        tmem_st8(pbase + 48, Q3);
                    }
                }
                if (do_tm) tmem_wait_st();
                tc_fence_before();
                mbar_arrive(&bars[B_P2]);
            }
            mbar_wait(&bars[B_ND2], ph_nd2); ph_nd2 ^= 1;   // every MMA of this tile is complete
            tc_fence_after();
            cp_async_wait<0>();
        }

        // ---- the CTA's accumulators -> its slab [2][N][KP] (grid <= n_tiles: every CTA had a tile) ----
        if (do_tm) {
            float* sa = slab + (size_t)(fr_ok ? fr : 0) * KP;
            float* sb = sa + (size_t)N * KP;
#pragma unroll
            for (int cg = 0; cg < 4; ++cg) {
                uint32_t a[16], bq[16];
                tmem_ld16(lane_base + T_ACC + 128 * half + 16 * cg, a);       // warp-collective: no lane predicate
                tmem_ld16(lane_base + T_ACC + 128 * half + 64 + 16 * cg, bq);
                tmem_wait_ld();
                if (fr_ok) {
#pragma unroll
                    for (int j = 0; j < 16; j += 4) {
                        *reinterpret_cast<uint4*>(sa + 16 * cg + j) = make_uint4(a[j], a[j + 1], a[j + 2], a[j + 3]);
                        *reinterpret_cast<uint4*>(sb + 16 * cg + j) = make_uint4(bq[j], bq[j + 1], bq[j + 2], bq[j + 3]);
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc(tmem, 512);
}

size_t tc_smem(int N, int NF, int nst) {
    return (size_t)3 * NF * 128 + 3 * HS_BYTES + (size_t)nst * 2 * N * SUBP * 4 + B_COUNT * 8 + 16;
}

}  // namespace

void nmf_tc_configure(nmf_plan* p) {
    p->t_ctas = 0; p->t_nst = 0;
    if (p->K > KP || p->N > 256) return;
    const int NF = (p->N + 31) / 32 * 32;
    int nst = 3;
    if (tc_smem(p->N, NF, nst) > 227 * 1024) nst = 2;
    if (tc_smem(p->N, NF, nst) > 227 * 1024) return;
    const long long n_tiles = (p->P + TILE - 1) / TILE;
    long long ctas = p->num_sms / p->batch;
    if (ctas < 1) ctas = 1;
    if (ctas > n_tiles) ctas = n_tiles;
    const long long per = (n_tiles + ctas - 1) / ctas;      // even out: every CTA gets `per` or one fewer
    ctas = (n_tiles + per - 1) / per;
    p->t_ctas = (int)ctas; p->t_nst = nst;
}

size_t nmf_tc_workspace(const nmf_plan* p) {
    if (!p->t_ctas) return 0;
    return (size_t)p->batch * p->t_ctas * 2 * p->N * KP * sizeof(float);
}

bool nmf_tc_available(const nmf_plan* p) { return p->t_ctas != 0; }

int nmf_tc_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters, int batch) {
    if (!p->t_ctas) return NMF_ERR_UNSUPPORTED;
    TcArgs a;
    a.X = X; a.Om = Om; a.W = W; a.H = H; a.slab = reinterpret_cast<float*>(p->ws);
    a.N = p->N; a.K = p->K; a.P = p->P; a.n_tiles = (p->P + TILE - 1) / TILE;
    a.NF = (p->N + 31) / 32 * 32; a.MT = (p->N + 127) / 128; a.KS = (p->K + 15) / 16;
    const size_t smem = tc_smem(p->N, a.NF, p->t_nst);
    if (!p->t_attr_done) {
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_tc_iter<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        NMF_CUDA_TRY(p, cudaFuncSetAttribute(k_tc_iter<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        p->t_attr_done = true;
    }
    const dim3 grid(p->t_ctas, batch);
    for (int it = 0; it < iters; ++it) {
        if (p->t_nst == 3) k_tc_iter<3><<<grid, CTA_THREADS, smem, p->stream>>>(a);
        else k_tc_iter<2><<<grid, CTA_THREADS, smem, p->stream>>>(a);
        p->launches++;
        int rc = nmf_launch_w_update(p, a.slab, W, p->N, p->K, KP, p->t_ctas, batch);
        if (rc) return rc;
    }
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

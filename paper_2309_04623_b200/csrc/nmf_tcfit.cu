// nmf_tcfit.cu -- fused per-pixel-tile NMF iteration on the tcgen05 tensor cores.
//
// One persistent, warp-specialised CTA per SM walks tiles of 128 pixels:
//   warps 0-7  element-wise warps, two groups of four (one thread per TMEM lane in each group)
//   warps 8-11 one MMA issuer (one elected thread issues every tcgen05.mma / tcgen05.commit), one TMA producer (one
//              thread streams H, X and Omega tiles through a ring of 16 KB slots) and two idle warps that wait at the
//              final barrier (384 threads get the same 168 registers as 320).  Whether the CTA carries the two
//              idle warps (PLACE = 1: 384 threads, roles on warps 11 / 10) or not (PLACE = 0: 320 threads, roles on
//              warps 8 / 9) is a template parameter chosen per shape on the host from measurements: with 384
//              threads every role assignment measured the same, the thread count is what matters
// All six contractions of Eq. 3 run as tcgen05.mma kind::f16 on BF16 operands with FP32
// accumulation in TMEM.  Every FP32 operand x is split exactly into three BF16 pieces x = x1 + x2 + x3
// (x1 = x to 8 significant bits, x2 = the next 8 bits, x3 = the rest) and a product a*b is evaluated as the six piece
// products a1b1 + a1b2 + a2b1 + a2b2 + a1b3 + a3b1 (dropped terms <= 2^-22 |ab|), so the arithmetic stays
// FP32-faithful ("BF16x3", the BF16 analogue of the 3xTF32 split; 16-bit operands can be read both K-major
// and MN-major from one no-swizzle buffer, so W and H' serve two contractions each from one copy).
//
// Per tile (p0 .. p0+127), with W (3 pieces, [frames][comps]) resident in shared memory:
//   H phase (TMEM lane = pixel), 16 frames per chunk, chunk c handled by group c & 1:
//     H0   the H tile (TMA -> ring) is split and written to shared memory as Hs[pixel][comp]       (a1)
//     S    S^T[pixel][frame] = Hs . Ws^T, 32 frames (two chunks) per series of SS MMAs              (a2)
//     EW   thread = (pixel, 16 frames): X, Omega from the ring; q = Om*X (select), r = Om*S,
//          split -> TMEM (R1, R2 overwrite S in place)                                              (a3)
//     ND   Num^T += Q^T . W, Den^T += R^T . W   (A from TMEM, B = MN-major view of Ws)              (a4)
//     UPD  h' = h * num / max(den, eps) -> global H and, split, back into Hs                        (a5)
//   W phase (TMEM lane = frame), one M tile of 128 frames at a time, 16 pixels per chunk, chunk c by group c & 1:
//     WT   the M tile's rows of the W pieces are staged into TMEM (tcgen05.st)
//     S'   S'[frame][pixel] = W . Hs^T, 32 pixels per series of TS MMAs (A = W tile in TMEM: tensor rate) (a6)
//     EW   thread = (frame, 16 pixels): X, Omega re-read (L2) through TMA (64-byte swizzled rows);
//          q, r' = Om*S' split -> TMEM                                                              (a6)
//     AB   A += Q . Hs, B += R' . Hs  (A from TMEM, B = MN-major view of Hs), accumulated in TMEM
//          over all tiles of the CTA                                                                (a7)
//   After the last tile the [2][N][64] accumulators go to this CTA's slab; nmf_launch_w_update reduces
//   the slabs in fixed order and updates W (a8).
// S / S' are double-buffered in TMEM per 32-frame / 32-pixel super-chunk and each group has its own piece columns, so
// the element-wise work of one buffer overlaps the MMAs of the other, and the TMA ring runs ahead across phase and
// tile borders.  In projection mode (nmf_project, a9) H is fixed and only H0 and the W phase run.
#include <cuda.h>
#include "nmf_common.cuh"
#include "nmf_tc.cuh"

namespace {
using namespace tc;

constexpr int EW_WARPS = 8;
// warps 8 .. 11: MMA issuer, TMA producer and two idle warps; which is which is a template parameter (PLACE)
constexpr int TILE = 128;                  // pixels per tile = UMMA M of the H phase
constexpr int FCH = 16;                    // frames per H-phase chunk (one UMMA K step)
constexpr int PCH = 16;                    // pixels per W-phase chunk
constexpr int NCH2 = TILE / PCH;           // W-phase chunks per tile
constexpr int KP = 64;                     // components padded to the MN-major N of stages 2 and 4
constexpr int HS_SB = 16 * 128;            // Hs: bytes between 8-component groups (128 pixels x 16 B)
constexpr int HS_BYTES = 8 * HS_SB;        // one BF16 piece of the H tile
constexpr int SLOT = 16384;                // ring slot bytes
constexpr int MAX_SLOTS = 8;
constexpr int FLUSH_TILES = 16;            // tiles accumulated in TMEM between two flushes of A / B into the slab

// TMEM columns (512 allocated).  A super-chunk is two chunks (32 frames / 32 pixels), one per group.
constexpr uint32_t T_NUM = 0, T_DEN = 64;  // H phase: Num^T, Den^T [pixel][64]
constexpr uint32_t T_HZ = 128;             //   Z[jb] at T_HZ + 32 jb: S of super-chunk j (jb = j & 1); group g owns columns
                                           //   16 g .. 16 g + 15 and overwrites them in place with R1 (8) and R2 (8)
constexpr uint32_t T_HE = 192;             //   E[g] at T_HE + 32 g: R3, Q1, Q2, Q3 (8 columns each), single-buffered
constexpr uint32_t T_WZ = 0;               // W phase, one 128-frame M tile at a time: Z[jb] at 32 jb (Num/Den are dead by then)
constexpr uint32_t T_WE = 64;              //   E[g] at T_WE + 32 g
constexpr uint32_t T_WT = 128;             //   the M tile's rows of W as TMEM A operand: piece i at T_WT + 32 i (comps 2c, 2c+1
                                           //   in column c), so the S' MMAs read A from TMEM and run at the tensor rate
constexpr uint32_t T_ACC = 256;            // A_acc[m] at T_ACC + 128 m, B_acc[m] at + 64 (persistent over tiles)

struct TcArgs {
    CUtensorMap mH;            // H   [B*K, P]  box [32 comps][128 px]
    CUtensorMap mXh, mOh;      // X, Om [B*N, P] box [16 frames][128 px]          (H phase)
    CUtensorMap mXw, mOw;      // X, Om [B*N, P] box [128 frames][16 px], 64-byte swizzle (W phase, one M tile)
    const float* W; float* H; float* slab;
    int N, K; long long P; long long n_tiles;
    int NF;                    // frames padded to a multiple of 16 (rows of the W pieces)
    int NC;                    // H-phase chunks = NF / 16
    int MT;                    // 128-frame M tiles of the W phase (1 or 2)
    int KH;                    // 32-component slots of the H tile (1 or 2)
    int NS;                    // ring slots
    int proj;                  // 1: projection (a9): H is fixed, only the W phase runs (X = targets, Om = omega, W = coef)
};

// mbarrier slots
enum { B_HS = 0, B_HS2, B_S0, B_S1, B_P0, B_P1, B_NDG0, B_NDG1, B_ND, B_S20, B_S21, B_P20, B_P21, B_ABG0, B_ABG1, B_AB, B_WT,
       B_FULL, B_EMPTY = B_FULL + MAX_SLOTS, B_COUNT = B_EMPTY + MAX_SLOTS };

template <int KS, int PLACE>
__global__ void __launch_bounds__(PLACE ? 384 : 320, 1)
k_tc_iter(const __grid_constant__ TcArgs g) {
    constexpr int W_MMA = PLACE ? 11 : 8, W_TMA = PLACE ? 10 : 9;
    constexpr int THREADS = PLACE ? 384 : 320;           // PLACE 1 adds two idle warps (8, 9)
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K, NF = g.NF, NC = g.NC, MT = g.MT, KH = g.KH;
    const uint32_t NS = (uint32_t)g.NS;
    const long long P = g.P;
    const int WS_SB = (NF / 8) * 128;                   // Ws: bytes between 8-component groups
    const int WS_BYTES = 8 * WS_SB;
    unsigned char* ws_p = smem;                         // 3 pieces of W
    unsigned char* hs_p = ws_p + 3 * WS_BYTES;          // 3 pieces of the H tile
    unsigned char* ring = hs_p + 3 * HS_BYTES;          // NS slots of 16 KB (1024-byte aligned)
    uint64_t* bars = reinterpret_cast<uint64_t*>(ring + (size_t)NS * SLOT);
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    float* __restrict__ H = g.H + (size_t)b * K * P;
    float* slab = g.slab + ((size_t)b * gridDim.x + blockIdx.x) * 2 * (size_t)N * KP;

    // ---------------- setup: barriers, TMEM, W pieces ----------------
    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_WARPS); mbar_init(&bars[B_HS2], EW_WARPS);
        mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1);
        mbar_init(&bars[B_P0], 4); mbar_init(&bars[B_P1], 4); mbar_init(&bars[B_ND], 1);
        mbar_init(&bars[B_NDG0], 1); mbar_init(&bars[B_NDG1], 1);
        mbar_init(&bars[B_S20], 1); mbar_init(&bars[B_S21], 1); mbar_init(&bars[B_WT], EW_WARPS);
        mbar_init(&bars[B_P20], 4); mbar_init(&bars[B_P21], 4); mbar_init(&bars[B_AB], 1);
        mbar_init(&bars[B_ABG0], 1); mbar_init(&bars[B_ABG1], 1);
        for (uint32_t s = 0; s < NS; ++s) { mbar_init(&bars[B_FULL + s], 1); mbar_init(&bars[B_EMPTY + s], EW_WARPS); }
        mbar_fence_init();
    }
    if (warp == W_MMA) tmem_alloc(tptr, 512);
    if (warp == W_TMA && lane == 0) {
        tma_prefetch_desc(&g.mH); tma_prefetch_desc(&g.mXh); tma_prefetch_desc(&g.mOh);
        tma_prefetch_desc(&g.mXw); tma_prefetch_desc(&g.mOw);
    }
    for (int i = tid; i < NF * 8; i += THREADS) {   // (frame n, component group kg): 8 values -> 3 x 16 B
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
    const uint32_t ws_s = smem_u32(ws_p), hs_s = smem_u32(hs_p), ring_s = smem_u32(ring);
    const bool proj = g.proj != 0;
    const int NCR = proj ? 0 : NC;                       // H-phase chunks (none in projection mode)
    const uint32_t slots_per_tile = (uint32_t)(KH + NCR + MT * NCH2);
    const uint32_t ns_magic = 0xffffffffu / NS + 1u;    // seq / NS == umulhi(seq, ns_magic) for seq < 2^29
    auto slot_of = [&](uint32_t seq, uint32_t& par) -> uint32_t {
        const uint32_t qd = __umulhi(seq, ns_magic);
        par = qd & 1u;
        return seq - qd * NS;
    };

    if (warp == W_TMA) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            uint32_t seq = 0;
            auto acquire = [&](uint32_t bytes) -> uint32_t {      // next ring slot, armed for `bytes`
                uint32_t par;
                const uint32_t s = slot_of(seq, par);
                mbar_wait(&bars[B_EMPTY + s], par ^ 1u);
                mbar_expect_tx(&bars[B_FULL + s], bytes);
                ++seq;
                return s;
            };
            for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
                const int p0 = (int)(tile * TILE);
                for (int h = 0; h < KH; ++h) {
                    const uint32_t s = acquire(32 * TILE * 4);
                    tma_load_2d(ring_s + s * SLOT, &g.mH, p0, b * K + 32 * h, &bars[B_FULL + s]);
                }
                for (int c = 0; c < NCR; ++c) {
                    const uint32_t s = acquire(2 * FCH * TILE * 4);
                    tma_load_2d(ring_s + s * SLOT, &g.mXh, p0, b * N + FCH * c, &bars[B_FULL + s]);
                    tma_load_2d(ring_s + s * SLOT + FCH * TILE * 4, &g.mOh, p0, b * N + FCH * c, &bars[B_FULL + s]);
                }
                for (int m = 0; m < MT; ++m)             // W phase: M tile m's 128 rows of X and Omega, 16 px at a time
                    for (int c = 0; c < NCH2; ++c) {
                        const uint32_t s = acquire(2 * 128 * PCH * 4);
                        tma_load_2d(ring_s + s * SLOT, &g.mXw, p0 + PCH * c, b * N + 128 * m, &bars[B_FULL + s]);
                        tma_load_2d(ring_s + s * SLOT + 128 * PCH * 4, &g.mOw, p0 + PCH * c, b * N + 128 * m, &bars[B_FULL + s]);
                    }
            }
        }
    } else if (warp == W_MMA) {
        // =========================== MMA issuer (whole warp converged; one elected lane issues) ===========================
        uint32_t ph = 0;                              // phase bits, indexed by barrier slot
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; tc_fence_after(); };
        constexpr uint32_t id_s32 = idesc_bf16(128, 32, 0), id_s16 = idesc_bf16(128, 16, 0), id_nd = idesc_bf16(128, 64, 1);
        // piece pairs (a, b), small products first: a1b3 a3b1 a2b2 a1b2 a2b1 a1b1
        constexpr int pa[6] = {0, 2, 1, 0, 1, 0}, pb[6] = {2, 0, 1, 1, 0, 0};
        uint64_t d_hs_k[3], d_hs_mn[3], d_ws_k[3], d_ws_mn[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            d_hs_k[i] = smem_desc(hs_s + i * HS_BYTES, HS_SB, 128);
            d_hs_mn[i] = smem_desc(hs_s + i * HS_BYTES, 128, HS_SB);
            d_ws_k[i] = smem_desc(ws_s + i * WS_BYTES, WS_SB, 128);
            d_ws_mn[i] = smem_desc(ws_s + i * WS_BYTES, 128, WS_SB);
        }
        const uint32_t ws_kstep = (uint32_t)(2 * WS_SB) >> 4;
        constexpr uint32_t hs_kstep = (uint32_t)(2 * HS_SB) >> 4;
        const int NSC = (NC + 1) / 2;                    // H-phase super-chunks of 32 frames (the last may hold 16)
        constexpr int NSC2 = NCH2 / 2;                   // W-phase super-chunks of 32 pixels
        uint32_t acc_started = 0, itm = 0;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, ++itm) {
            if (itm % FLUSH_TILES == 0) acc_started = 0;         // the accumulators were flushed into the slab
            // ---- H phase ----
            auto issue_S = [&](int j) {                  // S(j): [128 px] x [32 frames], K = comps -> Z[j & 1]
                if (elect_one()) {
                    const uint32_t d = tmem + T_HZ + 32 * (j & 1);
                    const uint32_t boff = (uint32_t)(j * 4 * 128) >> 4;
                    const uint32_t id = (2 * j + 1 < NC) ? id_s32 : id_s16;
#pragma unroll
                    for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                        for (int ks = 0; ks < KS; ++ks)
                            mma16_ss(d, d_hs_k[pa[pr]] + ks * hs_kstep, d_ws_k[pb[pr]] + boff + ks * ws_kstep, id,
                                     (pr | ks) ? 1u : 0u);
                    mma_commit(&bars[B_S0 + (j & 1)]);
                }
                __syncwarp();
            };
            wait(B_HS);
            if (!proj) {
            issue_S(0);
            if (NSC > 1) issue_S(1);
            for (int j = 0; j < NSC; ++j) {
                for (int gg = 0; gg < 2; ++gg) {
                    const int c = 2 * j + gg;
                    if (c >= NC) break;
                    wait(B_P0 + gg);
                    if (elect_one()) {
                        const uint32_t z = tmem + T_HZ + 32 * (j & 1) + 16 * gg, e = tmem + T_HE + 32 * gg;
                        const uint32_t a_q[3] = {e + O_Q1, e + O_Q2, e + O_Q3};
                        const uint32_t a_r[3] = {z, z + 8, e + O_R3};
                        const uint32_t boff = (uint32_t)(c * 2 * 128) >> 4;   // 16 frames = 2 row groups
#pragma unroll
                        for (int pr = 0; pr < 6; ++pr) {
                            const uint32_t acc = (c > 0 || pr > 0) ? 1u : 0u;
                            mma16_ts(tmem + T_NUM, a_q[pa[pr]], d_ws_mn[pb[pr]] + boff, id_nd, acc);
                            mma16_ts(tmem + T_DEN, a_r[pa[pr]], d_ws_mn[pb[pr]] + boff, id_nd, acc);
                        }
                        mma_commit(&bars[B_NDG0 + gg]);
                    }
                    __syncwarp();
                }
                if (j + 2 < NSC) issue_S(j + 2);
            }
            if (elect_one()) mma_commit(&bars[B_ND]);
            __syncwarp();
            }
            // ---- W phase: one 128-frame M tile at a time; A of S' = the tile's rows of W, staged in TMEM ----
            auto issue_S2 = [&](int j) {                 // S'(j): [128 frames] x [32 px], K = comps -> Z[j & 1]
                if (elect_one()) {
                    const uint32_t boff = (uint32_t)(j * 4 * 128) >> 4;
                    const uint32_t d = tmem + T_WZ + 32 * (j & 1);
#pragma unroll
                    for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                        for (int ks = 0; ks < KS; ++ks)
                            mma16_ts(d, tmem + T_WT + 32 * pa[pr] + 8 * ks, d_hs_k[pb[pr]] + boff + ks * hs_kstep,
                                     id_s32, (pr | ks) ? 1u : 0u);
                    mma_commit(&bars[B_S20 + (j & 1)]);
                }
                __syncwarp();
            };
            if (!proj) wait(B_HS2);                      // H' pieces in Hs and W tile 0 in TMEM are in place
            for (int m = 0; m < MT; ++m) {
                if (m > 0) wait(B_WT);                   // W tile m staged (every S' of tile m - 1 has completed)
                issue_S2(0);
                issue_S2(1);
                for (int j = 0; j < NSC2; ++j) {
                    for (int gg = 0; gg < 2; ++gg) {
                        const int c = 2 * j + gg;
                        wait(B_P20 + gg);
                        if (elect_one()) {
                            const uint32_t boff = (uint32_t)(c * 2 * 128) >> 4;   // 16 pixels = 2 row groups
                            const uint32_t z = tmem + T_WZ + 32 * (j & 1) + 16 * gg;
                            const uint32_t e = tmem + T_WE + 32 * gg;
                            const uint32_t a_q[3] = {e + O_Q1, e + O_Q2, e + O_Q3};
                            const uint32_t a_r[3] = {z, z + 8, e + O_R3};
#pragma unroll
                            for (int pr = 0; pr < 6; ++pr) {
                                const uint32_t acc = (((acc_started >> m) & 1u) || pr > 0) ? 1u : 0u;
                                mma16_ts(tmem + T_ACC + 128 * m, a_q[pa[pr]], d_hs_mn[pb[pr]] + boff, id_nd, acc);
                                mma16_ts(tmem + T_ACC + 128 * m + 64, a_r[pa[pr]], d_hs_mn[pb[pr]] + boff, id_nd, acc);
                            }
                            mma_commit(&bars[B_ABG0 + gg]);
                        }
                        __syncwarp();
                        acc_started |= 1u << m;
                    }
                    if (j + 2 < NSC2) issue_S2(j + 2);
                }
            }
            if (elect_one()) mma_commit(&bars[B_AB]);
            __syncwarp();
        }
    } else if (warp < EW_WARPS) {
        // =========================== element-wise warps ===========================
        const int q = warp & 3, grp = warp >> 2;
        const int t = 32 * q + lane;                     // TMEM lane: H-phase pixel / W-phase frame in the M tile
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; };
        auto wait_full = [&](uint32_t seq) -> const unsigned char* {
            uint32_t par;
            const uint32_t s = slot_of(seq, par);
            mbar_wait(&bars[B_FULL + s], par);
            return ring + (size_t)s * SLOT;
        };
        auto release = [&](uint32_t seq) {               // this warp is done reading the slot
            __syncwarp();
            uint32_t par;
            if (lane == 0) mbar_arrive(&bars[B_EMPTY + slot_of(seq, par)]);
        };
        auto warp_arrive = [&](int bar) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[bar]);
        };
        // An mbarrier wait tests a phase PARITY, so a warp may only test the "full" barrier of a slot for use u if it
        // also saw use u - 1 (a group that ran ahead of a late TMA load would see the parity of use u - 2 and read a
        // slot that has not landed).  Every element-wise warp therefore waits for and releases EVERY slot, in ring
        // order: the slots of the other group are only observed.
        auto observe = [&](uint32_t seq) { wait_full(seq); release(seq); };
        // rows 128 m .. 128 m + 127 of the W pieces -> TMEM (A operand of S'): group 0 stages pieces 0 and 1, group 1 piece 2
        auto stage_wt = [&](int m) {
            const int fr = 128 * m + t;
            const uint32_t rowoff = (uint32_t)((fr & 7) * 16 + (fr >> 3) * 128);
            for (int i = grp ? 2 : 0; i < (grp ? 3 : 2); ++i) {
                uint32_t v[32];
#pragma unroll
                for (int kg = 0; kg < 8; ++kg) {
                    uint4 w = make_uint4(0u, 0u, 0u, 0u);
                    if (fr < NF) w = *reinterpret_cast<const uint4*>(ws_p + i * WS_BYTES + rowoff + kg * WS_SB);
                    v[4 * kg] = w.x; v[4 * kg + 1] = w.y; v[4 * kg + 2] = w.z; v[4 * kg + 3] = w.w;
                }
                tmem_st32(lane_base + T_WT + 32 * i, v);
            }
            tmem_wait_st();
        };
        // The tensor cores accumulate in FP32 with truncation, so a long sum of positive terms comes out low and A, B do
        // not lose exactly the same fraction: accumulated over all tiles of a CTA, W <- W A / B was biased by 3e-6 per
        // iteration (8e-4 after 200 iterations at 200 x 1024^2, all of it in the scale split between W and H).  The
        // accumulators are therefore added into the CTA's slab [2][N][KP] every FLUSH_TILES tiles and restarted.
        // Group g handles M tile g; `add` = the slab already holds earlier flushes.
        auto flush = [&](bool add) {
            tc_fence_after();
            if (grp < MT) {
                const int fr = 128 * grp + t;
                const bool fr_ok = fr < N;
                float* sa = slab + (size_t)(fr_ok ? fr : 0) * KP;
                float* sb = sa + (size_t)N * KP;
#pragma unroll
                for (int cg = 0; cg < 4; ++cg) {
                    uint32_t a[16], bq[16];
                    tmem_ld16(lane_base + T_ACC + 128 * grp + 16 * cg, a);       // warp-collective: no lane predicate
                    tmem_ld16(lane_base + T_ACC + 128 * grp + 64 + 16 * cg, bq);
                    tmem_wait_ld();
                    if (fr_ok) {
#pragma unroll
                        for (int j = 0; j < 16; j += 4) {
                            float4 va = make_float4(__uint_as_float(a[j]), __uint_as_float(a[j + 1]), __uint_as_float(a[j + 2]), __uint_as_float(a[j + 3]));
                            float4 vb = make_float4(__uint_as_float(bq[j]), __uint_as_float(bq[j + 1]), __uint_as_float(bq[j + 2]), __uint_as_float(bq[j + 3]));
                            float4* pa = reinterpret_cast<float4*>(sa + 16 * cg + j);
                            float4* pb = reinterpret_cast<float4*>(sb + 16 * cg + j);
                            if (add) {
                                const float4 oa = *pa, ob = *pb;
                                va.x += oa.x; va.y += oa.y; va.z += oa.z; va.w += oa.w;
                                vb.x += ob.x; vb.y += ob.y; vb.z += ob.z; vb.w += ob.w;
                            }
                            *pa = va; *pb = vb;
                        }
                    }
                }
            }
            tc_fence_before();
        };
        uint32_t sq = 0;                                 // ring sequence number of this tile's first slot
        uint32_t itl = 0;                                // tiles of this CTA done
        bool first = true;
        const int NSC = (NC + 1) / 2;
        constexpr int NSC2 = NCH2 / 2;

        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, sq += slots_per_tile) {
            const long long p = tile * TILE + t;
            const bool p_ok = p < P;
            const long long pc = p_ok ? p : P - 1;

            // ---- H0: this group's 32 components of the H tile are split into Hs[pixel][comp] ----
            const float* hsl = nullptr;
            if (grp < KH) hsl = reinterpret_cast<const float*>(wait_full(sq + grp));
            uint32_t hp1[16], hp2[16], hp3[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int k0 = 32 * grp + 2 * j;         // pixels >= P arrive zero-filled
                const float h0 = (hsl && k0 < K) ? hsl[(2 * j) * TILE + t] : 0.f;
                const float h1 = (hsl && k0 + 1 < K) ? hsl[(2 * j + 1) * TILE + t] : 0.f;
                split3_pair(h0, h1, hp1[j], hp2[j], hp3[j]);
            }
            if (!first) { wait(B_AB); }                  // every MMA of the previous tile is complete: Hs is free
            if (!first && itl % FLUSH_TILES == 0) flush(itl > FLUSH_TILES);   // (the issuer restarts the accumulation with this
                                                         // tile; it waits for B_HS, which follows the flush)
            first = false;
            ++itl;
#pragma unroll
            for (int gq = 0; gq < 4; ++gq) {
                const uint32_t off = (t & 7) * 16 + (t >> 3) * 128 + (4 * grp + gq) * HS_SB;
                *reinterpret_cast<uint4*>(hs_p + off) = make_uint4(hp1[4 * gq], hp1[4 * gq + 1], hp1[4 * gq + 2], hp1[4 * gq + 3]);
                *reinterpret_cast<uint4*>(hs_p + HS_BYTES + off) = make_uint4(hp2[4 * gq], hp2[4 * gq + 1], hp2[4 * gq + 2], hp2[4 * gq + 3]);
                *reinterpret_cast<uint4*>(hs_p + 2 * HS_BYTES + off) = make_uint4(hp3[4 * gq], hp3[4 * gq + 1], hp3[4 * gq + 2], hp3[4 * gq + 3]);
            }
            if (grp < KH) release(sq + grp);
            if (1 - grp < KH) observe(sq + 1 - grp);
            if (proj) { stage_wt(0); tc_fence_before(); }        // (the previous tile's MMAs are complete: B_AB)
            fence_proxy_async();
            warp_arrive(B_HS);

            bool pending = false;                        // an ND / AB of this group may still be reading E[grp]
            if (!proj) {
            // ---- H phase: super-chunk j = chunks 2j (group 0) and 2j + 1 (group 1); thread = (pixel t, 16 frames) ----
            for (int j = 0; j < NSC; ++j) {
                const int c = 2 * j + grp;
                const bool have = c < NC;
                if (grp == 1) observe(sq + KH + c - 1);  // group 0's chunk of this super-chunk comes first in the ring
                float x[16], o[16];
                if (have) {
                    const uint32_t seq = sq + KH + c;
                    const float* xs = reinterpret_cast<const float*>(wait_full(seq));
                    const int nv = N - FCH * c;          // valid frames of this chunk (>= 16: all)
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        x[i] = xs[i * TILE + t];
                        o[i] = i < nv ? xs[FCH * TILE + i * TILE + t] : 0.f;
                    }
                }
                wait(B_S0 + (j & 1));                    // both groups track every completion of the buffer's barrier
                if (have) {
                    tc_fence_after();
                    const uint32_t zcol = lane_base + T_HZ + 32 * (j & 1) + 16 * grp;
                    uint32_t s[16], e[32];
                    tmem_ld16(zcol, s);
                    tmem_wait_ld();
                    ew16(x, o, s, zcol, e);
                    release(sq + KH + c);                // only now: every x, o value has been consumed (a release right
                                                         // after issuing the loads raced with the refill of the slot)
                    if (pending) { wait(B_NDG0 + grp); tc_fence_after(); }
                    tmem_st32(lane_base + T_HE + 32 * grp, e);
                    tmem_wait_st();
                    tc_fence_before();
                    warp_arrive(B_P0 + grp);
                    pending = true;
                }
                if (grp == 0 && c + 1 < NC) observe(sq + KH + c + 1);
            }
            // ---- UPD: h' = h * num / max(den, eps); thread = (pixel t, this group's 32 comps) ----
            // the old h is rebuilt exactly from its three BF16 pieces in Hs (h = h1 + h2 + h3, every partial sum exact)
            if (pending) wait(B_NDG0 + grp);
            wait(B_ND);                                  // Num, Den complete; every stage-1 read of Hs is done
            tc_fence_after();
            {
                float* hp = H + (size_t)(32 * grp) * P + pc;
#pragma unroll
                for (int gq = 0; gq < 4; ++gq) {
                    const int kg = 4 * grp + gq;
                    const uint32_t off = (t & 7) * 16 + (t >> 3) * 128 + kg * HS_SB;
                    uint32_t nm[8], dn[8];
                    tmem_ld8(lane_base + T_NUM + 8 * kg, nm);
                    tmem_ld8(lane_base + T_DEN + 8 * kg, dn);
                    const uint4 h1 = *reinterpret_cast<const uint4*>(hs_p + off);
                    const uint4 h2 = *reinterpret_cast<const uint4*>(hs_p + HS_BYTES + off);
                    const uint4 h3 = *reinterpret_cast<const uint4*>(hs_p + 2 * HS_BYTES + off);
                    const uint32_t a1[4] = {h1.x, h1.y, h1.z, h1.w}, a2[4] = {h2.x, h2.y, h2.z, h2.w}, a3[4] = {h3.x, h3.y, h3.z, h3.w};
                    tmem_wait_ld();
                    float hn[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j, hp += P) {
                        const int w = j >> 1;
                        const float hold = (j & 1)
                            ? (__uint_as_float(a1[w] & 0xffff0000u) + __uint_as_float(a2[w] & 0xffff0000u)) + __uint_as_float(a3[w] & 0xffff0000u)
                            : (__uint_as_float(a1[w] << 16) + __uint_as_float(a2[w] << 16)) + __uint_as_float(a3[w] << 16);
                        // padded comps / pixels carry h = 0 and num = 0: v = 0
                        const float v = __fdividef(hold * __uint_as_float(nm[j]), fmaxf(__uint_as_float(dn[j]), NMF_EPS));
                        if (p_ok && kg * 8 + j < K) *hp = v;
                        hn[j] = v;
                    }
                    uint32_t p1[4], p2[4], p3[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) split3_pair(hn[2 * j], hn[2 * j + 1], p1[j], p2[j], p3[j]);
                    *reinterpret_cast<uint4*>(hs_p + off) = make_uint4(p1[0], p1[1], p1[2], p1[3]);
                    *reinterpret_cast<uint4*>(hs_p + HS_BYTES + off) = make_uint4(p2[0], p2[1], p2[2], p2[3]);
                    *reinterpret_cast<uint4*>(hs_p + 2 * HS_BYTES + off) = make_uint4(p3[0], p3[1], p3[2], p3[3]);
                }
            }
            stage_wt(0);                                 // H-phase TMEM buffers are dead (B_ND): W tile 0 for S'
            fence_proxy_async();
            tc_fence_before();
            warp_arrive(B_HS2);
            }   // !proj

            // ---- W phase: M tile m, super-chunk j = chunks 2j + grp; thread = (frame 128 m + t, 16 pixels) ----
            pending = false;
            for (int m = 0; m < MT; ++m) {
                if (m > 0) {                             // this group's last S' wait of tile m - 1 is behind it: restage W
                    stage_wt(m);
                    tc_fence_before();
                    warp_arrive(B_WT);
                }
                const int fr = 128 * m + t;
                const bool active = 128 * m + 32 * q < N;            // warp-uniform: some lane has a frame
                for (int j = 0; j < NSC2; ++j) {
                    const int c = 2 * j + grp;
                    const uint32_t seq = sq + KH + NCR + NCH2 * m + c;
                    if (grp == 1) observe(seq - 1);
                    const unsigned char* xsl = wait_full(seq);       // X rows at +0, Omega rows at +8 KB
                    float x[16], o[16];
                    if (active) {
                        if (fr < N) {
                            const int sw = (t >> 1) & 3;
#pragma unroll
                            for (int ch = 0; ch < 4; ++ch) {
                                const float4 xv = *reinterpret_cast<const float4*>(xsl + t * 64 + ((ch ^ sw) << 4));
                                const float4 ov = *reinterpret_cast<const float4*>(xsl + 128 * PCH * 4 + t * 64 + ((ch ^ sw) << 4));
                                x[4 * ch] = xv.x; x[4 * ch + 1] = xv.y; x[4 * ch + 2] = xv.z; x[4 * ch + 3] = xv.w;
                                o[4 * ch] = ov.x; o[4 * ch + 1] = ov.y; o[4 * ch + 2] = ov.z; o[4 * ch + 3] = ov.w;
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < 16; ++i) { x[i] = 0.f; o[i] = 0.f; }
                        }
                    }
                    wait(B_S20 + (j & 1)); tc_fence_after();
                    uint32_t e[32];
                    if (active) {
                        const uint32_t zcol = lane_base + T_WZ + 32 * (j & 1) + 16 * grp;
                        uint32_t s[16];
                        tmem_ld16(zcol, s);
                        tmem_wait_ld();
                        ew16(x, o, s, zcol, e);
                    }
                    release(seq);                        // after the values were consumed (see the H phase)
                    if (pending) { wait(B_ABG0 + grp); tc_fence_after(); }
                    if (active) tmem_st32(lane_base + T_WE + 32 * grp, e);
                    tmem_wait_st();
                    tc_fence_before();
                    warp_arrive(B_P20 + grp);
                    pending = true;
                    if (grp == 0) observe(seq + 1);
                }
            }
            wait(B_ABG0 + grp);
        }
        wait(B_AB);                                      // every MMA of the last tile is complete
        flush(itl > FLUSH_TILES);                        // what was accumulated since the last flush (grid <= n_tiles: every
                                                         // CTA had a tile)
    }
    tc_fence_before();
    __syncthreads();
    if (warp == W_MMA) tmem_dealloc(tmem, 512);
}

constexpr size_t SMEM_MAX = 227 * 1024;

size_t tc_smem_fixed(int NF) { return (size_t)3 * NF * 128 + 3 * HS_BYTES + B_COUNT * 8 + 16; }

template <int KS, int PLACE>
cudaError_t launch_kp(const TcArgs& a, dim3 grid, size_t smem, cudaStream_t st, int device) {
    static bool attr_done[NMF_MAX_DEVICES] = {};                      // function attributes are per device
    if (device < 0 || device >= NMF_MAX_DEVICES || !attr_done[device]) {
        cudaError_t e = cudaFuncSetAttribute(k_tc_iter<KS, PLACE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
        if (e != cudaSuccess) return e;
        if (device >= 0 && device < NMF_MAX_DEVICES) attr_done[device] = true;
    }
    k_tc_iter<KS, PLACE><<<grid, PLACE ? 384 : 320, smem, st>>>(a);
    return cudaSuccess;
}
template <int KS>
cudaError_t launch_ks(const TcArgs& a, dim3 grid, size_t smem, cudaStream_t st, bool place, int device) {
    return place ? launch_kp<KS, 1>(a, grid, smem, st, device) : launch_kp<KS, 0>(a, grid, smem, st, device);
}

}  // namespace

void nmf_tc_configure(nmf_plan* p) {
    p->t_ctas = 0;
    if (p->K > KP || p->N > 256) return;
    if (p->P + TILE >= (1LL << 31) || (long long)p->batch * p->N >= (1LL << 31)) return;   // TMA coordinates are int32
    const int NF = (p->N + FCH - 1) / FCH * FCH;
    long long ns = ((long long)SMEM_MAX - (long long)tc_smem_fixed(NF)) / SLOT;
    if (ns > MAX_SLOTS) ns = MAX_SLOTS;
    if (ns < 4) return;
    const long long n_tiles = (p->P + TILE - 1) / TILE;
    long long ctas = p->num_sms / p->batch;
    if (ctas < 1) ctas = 1;
    if (ctas > n_tiles) ctas = n_tiles;
    const long long per = (n_tiles + ctas - 1) / ctas;      // even out: every CTA gets `per` or one fewer
    ctas = (n_tiles + per - 1) / per;
    p->t_ctas = (int)ctas;
}

size_t nmf_tc_workspace(const nmf_plan* p) {
    if (!p->t_ctas) return 0;
    const int prow = p->max_targets < 256 ? p->max_targets : 256;             // projection: <= 256 frames per pass
    const size_t fit = (size_t)p->batch * p->t_ctas * 2 * p->N * KP * sizeof(float);
    const size_t proj = (size_t)p->t_ctas * 2 * prow * KP * sizeof(float);
    return fit > proj ? fit : proj;
}

bool nmf_tc_available(const nmf_plan* p) { return p->t_ctas != 0; }

namespace {
// one launch sequence: `iters` x { fused tile kernel ; fixed-order reduce + update of W (or coef) }
int tc_run(nmf_plan* p, const float* X, const float* Om, float* W, const float* H, int rows, int iters, int batch, bool proj) {
    TcArgs a;
    const long long trows = (long long)batch * rows;
    if (!make_map(&a.mH, H, (long long)batch * p->K, p->P, 32, TILE, 0) ||
        !make_map(&a.mXh, X, trows, p->P, FCH, TILE, 0) || !make_map(&a.mOh, Om, trows, p->P, FCH, TILE, 0) ||
        !make_map(&a.mXw, X, trows, p->P, 128, PCH, 64) || !make_map(&a.mOw, Om, trows, p->P, 128, PCH, 64)) {
        if (!p->sticky) { p->sticky = NMF_ERR_CUDA; p->cuda_msg = "cuTensorMapEncodeTiled failed"; }
        return NMF_ERR_CUDA;
    }
    a.W = W; a.H = const_cast<float*>(H); a.slab = reinterpret_cast<float*>(p->ws);
    a.N = rows; a.K = p->K; a.P = p->P; a.n_tiles = (p->P + TILE - 1) / TILE;
    a.NF = (rows + FCH - 1) / FCH * FCH; a.NC = a.NF / FCH; a.MT = (rows + 127) / 128;
    a.KH = (p->K + 31) / 32; a.proj = proj ? 1 : 0;
    long long ns = ((long long)SMEM_MAX - (long long)tc_smem_fixed(a.NF)) / SLOT;
    a.NS = (int)(ns > MAX_SLOTS ? MAX_SLOTS : ns);
    const int KS = (p->K + 15) / 16;
    // CTA size, measured per shape on the box (same-box A/B, fit iteration): 320 threads (issuer / producer as warps
    // 8 / 9) win everywhere (survey batch -8 %, MIRI-shaped -6 %, K = 10 -4 %) except in the metric's own shape class
    // -- two M tiles with the last lane quadrant of the second one empty, four K steps -- where 384 threads (two
    // idle warps; any role assignment among warps 8 .. 11 measures the same) are 4 % faster.
    const bool place = a.MT == 2 && rows <= 224 && KS == 4;
    const size_t smem = tc_smem_fixed(a.NF) + (size_t)a.NS * SLOT;
    const dim3 grid(p->t_ctas, batch);
    int rc = nmf_run_iterations(p, proj ? 31 : 30, X, Om, W, H, nullptr, rows, batch, iters, [&]() -> int {
        cudaError_t e;
        switch (KS) {
            case 1: e = launch_ks<1>(a, grid, smem, p->stream, place, p->device); break;
            case 2: e = launch_ks<2>(a, grid, smem, p->stream, place, p->device); break;
            case 3: e = launch_ks<3>(a, grid, smem, p->stream, place, p->device); break;
            default: e = launch_ks<4>(a, grid, smem, p->stream, place, p->device); break;
        }
        NMF_CUDA_TRY(p, e);
        p->launches++;
        return nmf_launch_w_update(p, a.slab, W, rows, p->K, KP, p->t_ctas, batch);
    });
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}
}  // namespace

int nmf_tc_fit(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int iters, int batch) {
    if (!p->t_ctas) return NMF_ERR_UNSUPPORTED;
    return tc_run(p, X, Om, W, H, p->N, iters, batch, false);
}

// Projection (a9) on the tensor cores: the W phase alone with H fixed, X = targets, Omega = omega, W = coef.
// Frames are handled 256 at a time (the W phase holds two 128-row M tiles).
int nmf_tc_project(nmf_plan* p, const float* H, const float* T, const float* om, float* C, int M, int iters) {
    if (!p->t_ctas || !om) return NMF_ERR_UNSUPPORTED;
    for (int m0 = 0; m0 < M; m0 += 256) {
        const int rows = M - m0 < 256 ? M - m0 : 256;
        int rc = tc_run(p, T + (size_t)m0 * p->P, om + (size_t)m0 * p->P, C + (size_t)m0 * p->K, H, rows, iters, 1, true);
        if (rc) return rc;
    }
    return NMF_OK;
}

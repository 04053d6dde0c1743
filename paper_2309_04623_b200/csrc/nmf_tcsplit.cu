// nmf_tcsplit.cu -- the two half-steps of Eq. 3 as two persistent tcgen05 kernels, K <= 128.
//
// The fused kernel of nmf_tcfit.cu keeps Num/Den, S, the piece buffers AND the persistent W-phase accumulators
// of two 128-frame M tiles in the 512 TMEM columns: that leaves no column to feed the H-phase S stage from TMEM and
// room for only two chunks in flight between the element-wise warps and the tensor pipe.  The hand-over of a chunk
// (pieces stored -> mbarrier -> MMAs issued and executed -> commit -> mbarrier -> piece columns free) is a chain of
// fixed latencies that two chunks in flight do not cover: the tensor pipe sat idle half of the time.  Here the
// iteration is split, every kernel has TMEM to spare, and NG = 4 groups of element-wise warps keep four chunks in
// flight (NG = 2 where KP > 80 leaves no room):
//
//   k_tc_h<KS,NG>  H half-step (a1-a5).  TMEM lane = pixel.  The BF16 pieces of the H tile live in TMEM (as many of
//               the three as fit, the others in shared memory), so the S stage reads its A operand from TMEM and
//               runs at the tensor rate.  Num/Den take 2 KP columns, so KP = 16 KS goes up to 128 components.
//               W (3 BF16 pieces, [frames][comps]) is resident in shared memory.  The next tile's H pieces are
//               written as soon as the last S of a tile has completed, before the H update of that tile.
//   k_tc_w<KS,NG>  W half-step (a6-a7) with the new H.  TMEM lane = frame.  One 128-frame M tile per CTA
//               (blockIdx.z), so a CTA keeps 2 KP accumulator columns and its M tile's rows of W stay in TMEM for
//               the whole launch.  X and Omega rows are read only by the CTAs of their M tile; the ring is as deep
//               as shared memory allows (the kernel waited for data, not for the tensor pipe).  Also the projection kernel (a9) with
//               X = targets, Omega = omega, W = coef.
//   k_tc_wp<KS>    the same stages software-pipelined across tiles (two buffers of H pieces, S' of the next tile queued
//               behind AB of this one), K <= 64.  Used for projections of up to 64 frames, where it is 20 % faster; with
//               all 128 lanes busy the overlapped MMAs run 30 % slower and it loses to k_tc_w (see use_wp).
//   k_w_update_split   fixed-order fp64 reduction of the per-CTA slabs + W <- W o A / max(B, eps)  (a8)
//
// Ring slots and groups.  An mbarrier wait tests a phase PARITY, so a consumer may only test the "full" barrier of a
// slot for use u if it also consumed use u - 1 (a group that ran ahead of a late TMA load saw the parity of use
// u - 2 and read a slot that had not landed: tx-count corruption, launch failure at N = 200, K = 100, where the ring had
// three slots).  In k_tc_h work items are therefore dealt to the groups by their ring sequence number (item seq -> group
// seq % NG) and the number of slots is a multiple of NG: every use of a slot then belongs to the same group.  In k_tc_w
// (few, large slots) every element-wise warp waits for and releases every slot, in ring order, and reads only its own.
//
// X and Omega cross HBM twice per iteration instead of once (the fused kernel re-reads them through L2).
// Arithmetic and operand layouts are those of nmf_tcfit.cu (BF16x3 split, six piece products per product, FP32
// accumulation in TMEM, R1 / R2 written back over S in place).
#include <cuda.h>
#include "nmf_common.cuh"
#include "nmf_tc.cuh"

namespace {
using namespace tc;

constexpr int TILE = 128;                 // pixels per tile
constexpr int FCH = 16;                   // frames per H-step chunk (one UMMA K step)
constexpr int PCH = 16;                   // pixels per W-step chunk
constexpr int HS_SB = 16 * 128;           // [128 rows][comps] piece buffers: bytes between 8-component groups
constexpr int SLOT = 16384;               // k_tc_h ring slot: [16 frames][128 px] of X and of Omega, or [16 comps][128 px] of H
constexpr int PSW = 32;                   // k_tc_w: pixels per X / Omega ring slot (two W-step chunks)
constexpr int SLOTW = 32768;              // k_tc_w ring slot: [128 frames][32 px] of X and of Omega, or [64 comps][128 px] of H
constexpr int MAX_SLOTS = 12;
constexpr int MAX_NG = 4;
constexpr int FLUSH_TILES = 16;            // k_tc_w: tiles accumulated in TMEM between two flushes into the slab
constexpr size_t SMEM_MAX = 227 * 1024;

struct SplitArgs {
    CUtensorMap mH;            // H   [B*K, P]  box [16 comps][128 px] (k_tc_h) or [64 comps][128 px] (k_tc_w)
    CUtensorMap mX, mO;        // X, Om [B*rows, P]: box [16 frames][128 px] (k_tc_h) or [128 frames][32 px], 128-byte swizzle
                               // (k_tc_w: full 128-byte lines from HBM; 64-byte rows ran the kernel at a quarter of the HBM rate)
    const float* W; float* H; float* slab;
    int N, K; long long P; long long n_tiles;
    int NF;                    // frames padded to a multiple of 16
    int NC;                    // H-step chunks = NF / 16
    int NS;                    // ring slots
};

enum { B_HS = 0, B_UPD, B_S0, B_S1, B_DONE, B_HSB, B_DONEB, B_HFULL, B_FRDY = B_HFULL + 4, B_FDONE, B_P0, B_G0 = B_P0 + MAX_NG, B_FULL = B_G0 + MAX_NG,
       B_EMPTY = B_FULL + MAX_SLOTS, B_COUNT = B_EMPTY + MAX_SLOTS };

// piece pairs (a, b) of a product, small products first: a1b3 a3b1 a2b2 a1b2 a2b1 a1b1
__device__ constexpr int PA[6] = {0, 2, 1, 0, 1, 0}, PB[6] = {2, 0, 1, 1, 0, 0};

// pieces of the TMEM-resident A operand of the S stage that fit beside `fixed` columns and NG groups' S / E columns
__host__ __device__ constexpr int npt_of(int KP, int NG, int fixed) {
    const int room = 512 - fixed - 64 * NG;
    return room >= 3 * KP / 2 ? 3 : room >= KP ? 2 : room >= KP / 2 ? 1 : 0;
}

struct RingCtl {                          // ring slot arithmetic shared by producer and consumers
    uint32_t NS, magic;
    __device__ uint32_t slot(uint32_t seq, uint32_t& par) const {
        const uint32_t qd = __umulhi(seq, magic);      // seq / NS for seq < 2^29
        par = qd & 1u;
        return seq - qd * NS;
    }
};

__device__ __forceinline__ void st_piece_smem(unsigned char* base, int t, int kg, const uint32_t* w) {
    *reinterpret_cast<uint4*>(base + (t & 7) * 16 + (t >> 3) * 128 + kg * HS_SB) = make_uint4(w[0], w[1], w[2], w[3]);
}
// 16 components (rows of a ring slot, 128 floats apart) of pixel `t`, components kb .. kb + 15 -> three arrays of 8
// words; rows at or beyond K hold another problem's data (batched H) or zeros: they are replaced by zeros
__device__ __forceinline__ void split_rows16(const float* sl, int kb, int K, float* keep, uint32_t (&p1)[8], uint32_t (&p2)[8],
                                             uint32_t (&p3)[8]) {
    float h[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) h[j] = sl[j * TILE];                         // pixels >= P arrive zero-filled
    if (kb + 16 > K) {                                                        // rare: the last, partly filled block
#pragma unroll
        for (int j = 0; j < 16; ++j) if (kb + j >= K) h[j] = 0.f;
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        if (keep) { keep[2 * j] = h[2 * j]; keep[2 * j + 1] = h[2 * j + 1]; }
        split3_pair(h[2 * j], h[2 * j + 1], p1[j], p2[j], p3[j]);
    }
}

// =====================================================================================================================
// H half-step
// =====================================================================================================================
template <int KS, int NG>
__global__ void __launch_bounds__(32 * (4 * NG + 2), 1)
k_tc_h(const __grid_constant__ SplitArgs g) {
    constexpr int KP = 16 * KS;
    constexpr int EW_WARPS = 4 * NG, W_MMA = EW_WARPS, W_TMA = EW_WARPS + 1, THREADS = 32 * (EW_WARPS + 2);
    constexpr int NPT = npt_of(KP, NG, 2 * KP);                           // H pieces kept in TMEM
    constexpr uint32_t T_NUM = 0, T_DEN = KP, T_HT = 2 * KP;              // piece i of the H tile at T_HT + i KP / 2
    constexpr uint32_t T_Z = 2 * KP + NPT * KP / 2, T_E = T_Z + 32 * NG;  // Z[jb] at T_Z + 16 NG jb, E[g] at T_E + 32 g
    static_assert(T_E + 32 * NG <= 512, "TMEM");
    constexpr int NBLK = KP / 16;                        // 16-component blocks = H slots per tile
    constexpr int NB = (NBLK + NG - 1) / NG;             // blocks per group
    constexpr int HS_BYTES = (KP / 8) * HS_SB;           // one BF16 piece of the H tile in shared memory
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K, NF = g.NF, NC = g.NC;
    const long long P = g.P;
    const int WS_SB = (NF / 8) * 128;                   // Ws: bytes between 8-component groups
    const int WS_BYTES = (KP / 8) * WS_SB;
    unsigned char* ring = smem;                         // NS slots of 16 KB
    unsigned char* ws_p = ring + (size_t)g.NS * SLOT;   // 3 pieces of W
    unsigned char* hsx_p = ws_p + 3 * WS_BYTES;         // pieces NPT .. 2 of the H tile (those not in TMEM)
    uint64_t* bars = reinterpret_cast<uint64_t*>(hsx_p + (3 - NPT) * HS_BYTES);
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);
    const RingCtl rc{(uint32_t)g.NS, 0xffffffffu / (uint32_t)g.NS + 1u};

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y;
    NMF_TRC_DECL;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    float* __restrict__ H = g.H + (size_t)b * K * P;

    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_WARPS); mbar_init(&bars[B_UPD], EW_WARPS);
        mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1); mbar_init(&bars[B_DONE], 1);
        for (int i = 0; i < NG; ++i) { mbar_init(&bars[B_P0 + i], 4); mbar_init(&bars[B_G0 + i], 1); }
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
    const uint32_t ws_s = smem_u32(ws_p), hsx_s = smem_u32(hsx_p), ring_s = smem_u32(ring);
    const uint32_t slots_per_tile = (uint32_t)(NBLK + NC);
    const int NSC = (NC + NG - 1) / NG;                  // super-chunks of 16 NG frames (the last may hold fewer)

    if (warp == W_TMA) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            uint32_t seq = 0;
            auto acquire = [&](uint32_t bytes) -> uint32_t {      // next ring slot, armed for `bytes`
                uint32_t par;
                const uint32_t s = rc.slot(seq, par);
                mbar_wait(&bars[B_EMPTY + s], par ^ 1u);
                mbar_expect_tx(&bars[B_FULL + s], bytes);
                ++seq;
                return s;
            };
            // (bringing the data of the tiles ahead into L2 -- cp.async.bulk.prefetch.tensor a tile at a time or item by
            // item, or plain prefetch.global.L2 instructions from an extra warp -- made both kernels 20 - 50 % slower
            // on the box and was dropped)
            for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
                const int p0 = (int)(tile * TILE);
                for (int h = 0; h < NBLK; ++h) {
                    const uint32_t s = acquire(16 * TILE * 4);
                    tma_load_2d(ring_s + s * SLOT, &g.mH, p0, b * K + 16 * h, &bars[B_FULL + s]);
                }
                for (int c = 0; c < NC; ++c) {
                    const uint32_t s = acquire(2 * FCH * TILE * 4);
                    tma_load_2d(ring_s + s * SLOT, &g.mX, p0, b * N + FCH * c, &bars[B_FULL + s]);
                    tma_load_2d(ring_s + s * SLOT + FCH * TILE * 4, &g.mO, p0, b * N + FCH * c, &bars[B_FULL + s]);
                }
            }
        }
    } else if (warp == W_MMA) {
        // =========================== MMA issuer (whole warp converged; one elected lane issues) ===========================
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; tc_fence_after(); };
        constexpr uint32_t id_nd = idesc_bf16(128, KP, 1);
        uint64_t d_ws_k[3], d_ws_mn[3], d_hsx_k[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            d_ws_k[i] = smem_desc(ws_s + i * WS_BYTES, WS_SB, 128);
            d_ws_mn[i] = smem_desc(ws_s + i * WS_BYTES, 128, WS_SB);
            d_hsx_k[i] = smem_desc(hsx_s + (i >= NPT ? i - NPT : 0) * HS_BYTES, HS_SB, 128);
        }
        const uint32_t ws_kstep = (uint32_t)(2 * WS_SB) >> 4;
        constexpr uint32_t hs_kstep = (uint32_t)(2 * HS_SB) >> 4;
        bool first = true;
        uint32_t sq = 0;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, sq += slots_per_tile) {
            const int og = (int)((sq + NBLK) & (NG - 1));        // chunk c of this tile belongs to group (og + c) % NG
            auto issue_S = [&](int j) {                  // S(j): [128 px] x [16 NG frames], K = comps -> Z[j & 1]
                if (elect_one()) {
                    const uint32_t d = tmem + T_Z + 16 * NG * (j & 1);
                    const uint32_t boff = (uint32_t)(j * NG * 2 * 128) >> 4;      // 16 frames = 2 row groups of 128 bytes
                    const int nch = NC - NG * j < NG ? NC - NG * j : NG;
                    const uint32_t id = idesc_bf16(128, 16 * nch, 0);
#pragma unroll
                    for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                        for (int ks = 0; ks < KS; ++ks) {
                            const uint64_t bd = d_ws_k[PB[pr]] + boff + ks * ws_kstep;
                            if (PA[pr] < NPT) mma16_ts(d, tmem + T_HT + PA[pr] * (KP / 2) + 8 * ks, bd, id, (pr | ks) ? 1u : 0u);
                            else mma16_ss(d, d_hsx_k[PA[pr]] + ks * hs_kstep, bd, id, (pr | ks) ? 1u : 0u);
                        }
                    mma_commit(&bars[B_S0 + (j & 1)]);
                }
                __syncwarp();
            };
            wait(B_HS);
            NMF_TRC(TR_M_HS, 0);
            issue_S(0);
            if (NSC > 1) issue_S(1);
            NMF_TRC(TR_M_S, 1);
            if (!first) wait(B_UPD);                     // the previous tile's update has read Num / Den
            first = false;
            for (int j = 0; j < NSC; ++j) {
                for (int gi = 0; gi < NG; ++gi) {            // gi: position of the chunk in its super-chunk
                    const int c = NG * j + gi;
                    if (c >= NC) break;
                    const int gg = (og + gi) & (NG - 1);     // the group that prepares this chunk
                    wait(B_P0 + gg);
                    NMF_TRC(TR_M_READY, c);
                    if (elect_one()) {
                        const uint32_t z = tmem + T_Z + 16 * NG * (j & 1) + 16 * gi, e = tmem + T_E + 32 * gg;
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
                    NMF_TRC(TR_M_ISSUED, c);
                }
                if (j + 2 < NSC) { issue_S(j + 2); NMF_TRC(TR_M_S, j + 2); }
            }
            if (elect_one()) mma_commit(&bars[B_DONE]);
            __syncwarp();
        }
    } else if (warp < EW_WARPS) {
        // =========================== element-wise warps: group grp = warp / 4, lane quadrant q = warp % 4 ===========================
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
        // H0: the pieces of a tile's H -> TMEM / shared memory (A operand of S); a group takes the 16-component blocks
        // (one ring slot each) whose ring sequence number sqt + bi is its own modulo NG, and keeps their fp32 values
        // for the update
        auto h0 = [&](uint32_t sqt, float (&hv)[NB][16]) {
            NMF_TRC(TR_H0_BEGIN, 0);
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) {
                const int bi = (int)((grp - sqt) & (NG - 1)) + NG * bb;
                if (bi < NBLK) {
                    const float* hsl = reinterpret_cast<const float*>(wait_full(sqt + bi)) + t;
                    uint32_t p[3][8];
                    split_rows16(hsl, 16 * bi, K, hv[bb], p[0], p[1], p[2]);
                    release(sqt + bi);
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
                        if (i < NPT) tmem_st8(lane_base + T_HT + i * (KP / 2) + 8 * bi, p[i]);
                        else {
                            st_piece_smem(hsx_p + (i - NPT) * HS_BYTES, t, 2 * bi, &p[i][0]);
                            st_piece_smem(hsx_p + (i - NPT) * HS_BYTES, t, 2 * bi + 1, &p[i][4]);
                        }
                    }
                }
            }
            tmem_wait_st();
            if (NPT < 3) fence_proxy_async();
            tc_fence_before();
            warp_arrive(B_HS);
            NMF_TRC(TR_H0_END, 0);
        };
        float hold[NB][16];
        uint32_t sq = 0;
        h0(0, hold);
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, sq += slots_per_tile) {
            // ---- steps: this group's chunk of super-chunk j is NG j + zp (its ring slot has the group's sequence
            // number modulo NG); thread = (pixel t, 16 frames), two halves of 8 ----
            bool pending = false;
            const int zp = (int)((grp - (sq + NBLK)) & (NG - 1));
            for (int j = 0; j < NSC; ++j) {
                const int c = NG * j + zp;
                const bool have = c < NC;
                const float* xs = nullptr;
                if (have) xs = reinterpret_cast<const float*>(wait_full(sq + NBLK + c)) + t;
                NMF_TRC(TR_FULL, c);
                wait(B_S0 + (j & 1));                    // every group tracks every completion of the buffer's barrier
                NMF_TRC(TR_S, c);
                if (have) {
                    tc_fence_after();
                    const uint32_t zcol = lane_base + T_Z + 16 * NG * (j & 1) + 16 * zp;
                    const uint32_t ecol = lane_base + T_E + 32 * grp;
                    const int nv = N - FCH * c;          // valid frames of this chunk (>= 16: all)
                    uint32_t s[16];
                    tmem_ld16(zcol, s);
                    tmem_wait_ld();
                    NMF_TRC(TR_LD, c);
                    if (pending) { wait(B_G0 + grp); tc_fence_after(); }      // this group's E columns are free again
                    NMF_TRC(TR_EFREE, c);
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        float x[8], o[8];
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            x[i] = xs[(8 * hf + i) * TILE];
                            o[i] = xs[FCH * TILE + (8 * hf + i) * TILE];
                        }
                        if (nv < 16) {                   // rare: frames past N (another problem's rows in a batch)
#pragma unroll
                            for (int i = 0; i < 8; ++i) if (8 * hf + i >= nv) o[i] = 0.f;
                        }
                        Ew8 w;
                        ew8(x, o, &s[8 * hf], w);
                        ew8_store(zcol, ecol, hf, w);
                    }
                    release(sq + NBLK + c);              // after the values were consumed
                    tmem_wait_st();
                    tc_fence_before();
                    warp_arrive(B_P0 + grp);
                    NMF_TRC(TR_HANDED, c);
                    pending = true;
                }
            }
            // ---- every S of this tile has completed (each warp waited for all of them): the next tile's H pieces ----
            // (only where a thread keeps one block of 16 values: two live sets of NB x 16 registers would spill)
            constexpr bool EARLY = NB == 1;
            float hnext[NB][16];
            const bool has_next = tile + gridDim.x < g.n_tiles;
            if constexpr (EARLY) { if (has_next) h0(sq + slots_per_tile, hnext); }
            // ---- update: h' = h * num / max(den, eps) in place; thread = (pixel t, the components it split in H0) ----
            if (pending) wait(B_G0 + grp);
            wait(B_DONE);                                // Num, Den complete
            tc_fence_after();
            NMF_TRC(TR_UPD_BEGIN, 0);
            const long long p = tile * TILE + t;
            const bool p_ok = p < P;
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) {
                const int kb = 16 * ((int)((grp - sq) & (NG - 1)) + NG * bb);    // the blocks this thread split in H0
                if (kb < KP) {                           // (warp-uniform: tcgen05.ld is warp-collective)
                    uint32_t nm[16], dn[16];
                    tmem_ld16(lane_base + T_NUM + kb, nm);
                    tmem_ld16(lane_base + T_DEN + kb, dn);
                    tmem_wait_ld();
                    float* hp = H + (size_t)kb * P + (p_ok ? p : 0);
                    const int kv = p_ok ? K - kb : 0;    // components of this block that exist (none for a pixel past P)
#pragma unroll
                    for (int j = 0; j < 16; ++j, hp += P) {
                        const float v = __fdividef(hold[bb][j] * __uint_as_float(nm[j]), fmaxf(__uint_as_float(dn[j]), NMF_EPS));
                        if (j < kv) *hp = v;
                    }
                }
            }
            tc_fence_before();
            warp_arrive(B_UPD);
            NMF_TRC(TR_UPD_END, 0);
            if (has_next) {
                if constexpr (EARLY) {
#pragma unroll
                    for (int j = 0; j < 16; ++j) hold[0][j] = hnext[0][j];
                } else h0(sq + slots_per_tile, hold);
            }
        }
    }
    NMF_TRC_FLUSH(0);
    tc_fence_before();
    __syncthreads();
    if (warp == W_MMA) tmem_dealloc(tmem, 512);
}

// =====================================================================================================================
// W half-step (and projection)
// =====================================================================================================================
template <int KS, int NG>
__global__ void __launch_bounds__(32 * (4 * NG + 2), 1)
k_tc_w(const __grid_constant__ SplitArgs g) {
    constexpr int KP = 16 * KS;
    constexpr int EW_WARPS = 4 * NG, W_MMA = EW_WARPS, W_TMA = EW_WARPS + 1;
    constexpr int NPT = npt_of(KP, NG, 2 * KP);                           // W pieces of the M tile kept in TMEM
    constexpr uint32_t T_WT = 0;                                          // piece i at i KP / 2
    constexpr uint32_t T_Z = NPT * KP / 2, T_E = T_Z + 32 * NG;           // Z[jb] at T_Z + 16 NG jb, E[g] at T_E + 32 g
    constexpr uint32_t T_ACC = 512 - 2 * KP;                              // A at T_ACC, B at T_ACC + KP
    static_assert(T_E + 32 * NG <= T_ACC, "TMEM");
    constexpr int NBLK = KP / 16;                        // 16-component blocks
    constexpr int NHS = (NBLK + 3) / 4;                  // H ring slots (64 components each) per tile
    constexpr int NSW = TILE / PSW;                      // X / Omega ring slots per tile
    constexpr int NSC2 = TILE / (PCH * NG);              // super-chunks of 16 NG pixels per tile
    constexpr int HS_BYTES = (KP / 8) * HS_SB;           // one BF16 piece of the H tile / of the M tile's W rows
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K;
    unsigned char* ring = smem;
    unsigned char* hs_p = ring + (size_t)g.NS * SLOTW;  // 3 pieces of the H tile, [pixel][comp]
    unsigned char* wsx_p = hs_p + 3 * HS_BYTES;         // pieces NPT .. 2 of this M tile's rows of W
    uint64_t* bars = reinterpret_cast<uint64_t*>(wsx_p + (3 - NPT) * HS_BYTES);
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);
    const RingCtl rc{(uint32_t)g.NS, 0xffffffffu / (uint32_t)g.NS + 1u};

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y, m = blockIdx.z;
    NMF_TRC_DECL;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    // slab of this CTA: [B][MT][ctas][2][128][KP]
    float* slab = g.slab + (((size_t)b * gridDim.z + m) * gridDim.x + blockIdx.x) * 2 * (size_t)128 * KP;

    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_WARPS); mbar_init(&bars[B_UPD], 1);     // B_UPD: every MMA of the launch is complete
        mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1); mbar_init(&bars[B_DONE], 1);
        for (int i = 0; i < NG; ++i) { mbar_init(&bars[B_P0 + i], 4); mbar_init(&bars[B_G0 + i], 1); }
        // every element-wise warp waits for and releases EVERY ring slot (see "Ring slots and groups")
        for (int s = 0; s < g.NS; ++s) { mbar_init(&bars[B_FULL + s], 1); mbar_init(&bars[B_EMPTY + s], EW_WARPS); }
        mbar_fence_init();
    }
    if (warp == W_MMA) tmem_alloc(tptr, 512);
    if (warp == W_TMA && lane == 0) { tma_prefetch_desc(&g.mH); tma_prefetch_desc(&g.mX); tma_prefetch_desc(&g.mO); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tptr;
    const uint32_t hs_s = smem_u32(hs_p), wsx_s = smem_u32(wsx_p), ring_s = smem_u32(ring);
    const uint32_t slots_per_tile = (uint32_t)(NHS + NSW);

    if (warp < EW_WARPS) {
        // the M tile's rows of W -> TMEM / shared memory (A operand of S', fixed for the launch); lane = frame 128 m + t;
        // group g takes the 16-component blocks g, g + NG, ...
        const int q = warp & 3, grp = warp >> 2, t = 32 * q + lane;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const int fr = 128 * m + t;
        for (int bi = grp; bi < NBLK; bi += NG) {
            uint32_t p[3][8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int k0 = 16 * bi + 2 * j;
                const float w0 = (fr < N && k0 < K) ? W[(size_t)fr * K + k0] : 0.f;
                const float w1 = (fr < N && k0 + 1 < K) ? W[(size_t)fr * K + k0 + 1] : 0.f;
                split3_pair(w0, w1, p[0][j], p[1][j], p[2][j]);
            }
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                if (i < NPT) tmem_st8(lane_base + T_WT + i * (KP / 2) + 8 * bi, p[i]);
                else {
                    st_piece_smem(wsx_p + (i - NPT) * HS_BYTES, t, 2 * bi, &p[i][0]);
                    st_piece_smem(wsx_p + (i - NPT) * HS_BYTES, t, 2 * bi + 1, &p[i][4]);
                }
            }
        }
        tmem_wait_st();
        if (NPT < 3) fence_proxy_async();
        tc_fence_before();
    }
    __syncthreads();
    tc_fence_after();

    // Ring order per tile: the H tile (NHS slots of 64 components), then the M tile's rows of X and Omega, 32 pixels
    // (two chunks) per slot.  The ring is as deep as shared memory allows (five 32 KB slots at K <= 64: one tile ahead):
    // with four slots, half of them half empty, the element-wise warps waited 3000 cycles per tile for data.
    if (warp == W_TMA) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            uint32_t seq = 0;
            auto acquire = [&](uint32_t bytes) -> uint32_t {
                uint32_t par;
                const uint32_t s = rc.slot(seq, par);
                mbar_wait(&bars[B_EMPTY + s], par ^ 1u);
                mbar_expect_tx(&bars[B_FULL + s], bytes);
                ++seq;
                return s;
            };
            for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x) {
                const int p0 = (int)(tile * TILE);
                for (int h = 0; h < NHS; ++h) {
                    const uint32_t s = acquire(SLOTW);
                    NMF_TRCW(TR_T_ACQ, h);
                    tma_load_2d(ring_s + s * SLOTW, &g.mH, p0, b * K + 64 * h, &bars[B_FULL + s]);
                }
                for (int c = 0; c < NSW; ++c) {
                    const uint32_t s = acquire(SLOTW);
                    NMF_TRCW(TR_T_ACQ, NHS + c);
                    tma_load_2d(ring_s + s * SLOTW, &g.mX, p0 + PSW * c, b * N + 128 * m, &bars[B_FULL + s]);
                    tma_load_2d(ring_s + s * SLOTW + 128 * PSW * 4, &g.mO, p0 + PSW * c, b * N + 128 * m, &bars[B_FULL + s]);
                }
            }
        }
    } else if (warp == W_MMA) {
        // =========================== MMA issuer ===========================
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; tc_fence_after(); };
        constexpr uint32_t id_s = idesc_bf16(128, 16 * NG, 0), id_ab = idesc_bf16(128, KP, 1);
        uint64_t d_hs_k[3], d_hs_mn[3], d_wsx_k[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            d_hs_k[i] = smem_desc(hs_s + i * HS_BYTES, HS_SB, 128);
            d_hs_mn[i] = smem_desc(hs_s + i * HS_BYTES, 128, HS_SB);
            d_wsx_k[i] = smem_desc(wsx_s + (i >= NPT ? i - NPT : 0) * HS_BYTES, HS_SB, 128);
        }
        constexpr uint32_t hs_kstep = (uint32_t)(2 * HS_SB) >> 4;
        auto issue_S2 = [&](int j) {                     // S'(j): [128 frames] x [16 NG px], K = comps -> Z[j & 1]
            if (elect_one()) {
                const uint32_t boff = (uint32_t)(j * NG * 2 * 128) >> 4;
                const uint32_t d = tmem + T_Z + 16 * NG * (j & 1);
#pragma unroll
                for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                    for (int ks = 0; ks < KS; ++ks) {
                        const uint64_t bd = d_hs_k[PB[pr]] + boff + ks * hs_kstep;
                        if (PA[pr] < NPT) mma16_ts(d, tmem + T_WT + PA[pr] * (KP / 2) + 8 * ks, bd, id_s, (pr | ks) ? 1u : 0u);
                        else mma16_ss(d, d_wsx_k[PA[pr]] + ks * hs_kstep, bd, id_s, (pr | ks) ? 1u : 0u);
                    }
                mma_commit(&bars[B_S0 + (j & 1)]);
            }
            __syncwarp();
        };
        bool acc_started = false;
        uint32_t it = 0;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, ++it) {
            if (it % FLUSH_TILES == 0) acc_started = false;      // the accumulators were flushed into the slab (see below)
            wait(B_HS);                                  // the tile's H pieces are in Hs
            NMF_TRCW(TR_M_HS, 0);
            issue_S2(0);
            issue_S2(1);
            NMF_TRCW(TR_M_S, 1);
            for (int j = 0; j < NSC2; ++j) {
                for (int gg = 0; gg < NG; ++gg) {
                    const int c = NG * j + gg;
                    wait(B_P0 + gg);
                    NMF_TRCW(TR_M_READY, c);
                    if (elect_one()) {
                        const uint32_t boff = (uint32_t)(c * 2 * 128) >> 4;   // 16 pixels = 2 row groups
                        const uint32_t z = tmem + T_Z + 16 * NG * (j & 1) + 16 * gg, e = tmem + T_E + 32 * gg;
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
                    NMF_TRCW(TR_M_ISSUED, c);
                    acc_started = true;
                }
                if (j + 2 < NSC2) { issue_S2(j + 2); NMF_TRCW(TR_M_S, j + 2); }
            }
            if (elect_one()) mma_commit(&bars[B_DONE]);  // every MMA of this tile is complete: Hs may be rewritten
            __syncwarp();
        }
    } else if (warp < EW_WARPS) {
        // =========================== element-wise warps: group grp = warp / 4, lane quadrant q = warp % 4 ===========================
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
        // H0: the (new) H tile is split into Hs[pixel][comp]; thread = pixel t; ring slot h holds the components
        // 64 h .. 64 h + 63, group g takes the block of 16 components g of it (block g % 4 with two groups: two each)
        auto h0 = [&](uint32_t sqt) {
            NMF_TRCW(TR_H0_BEGIN, 0);
            for (int h = 0; h < NHS; ++h) {
                const float* hsl = reinterpret_cast<const float*>(wait_full(sqt + h)) + t;
                NMF_TRCW(TR_HSLOT, h);
                for (int sb = grp; sb < 4; sb += NG) {
                    const int bi = 4 * h + sb;
                    if (bi < NBLK) {
                        uint32_t p[3][8];
                        split_rows16(hsl + (16 * sb) * TILE, 16 * bi, K, nullptr, p[0], p[1], p[2]);
#pragma unroll
                        for (int i = 0; i < 3; ++i) {
                            st_piece_smem(hs_p + i * HS_BYTES, t, 2 * bi, &p[i][0]);
                            st_piece_smem(hs_p + i * HS_BYTES, t, 2 * bi + 1, &p[i][4]);
                        }
                    }
                }
                release(sqt + h);
            }
            fence_proxy_async();
            warp_arrive(B_HS);
            NMF_TRCW(TR_H0_END, 0);
        };
        // The tensor cores accumulate in FP32 with truncation: a sum of n positive terms comes out low by about n / 4
        // ulp, and A and B do not lose exactly the same fraction.  Accumulated over all ~110 tiles of a CTA, W <- W A / B
        // was biased by 1e-5 per iteration, the same sign for every component: after 200 iterations at 200 x 1024^2 W was
        // 1.6e-3 too large and H 1.6e-3 too small against the fp64 oracle (their product, and the cost, agreed to 1e-6;
        // the scale split between W and H is a neutral direction of Eq. 3 that nothing pulls back).  The accumulators are
        // therefore added into the CTA's slab [2][128][KP] every FLUSH_TILES tiles (FP32 adds, round to nearest, in a
        // fixed order) and restarted: the bias is proportional to the accumulation depth.  Group g handles the
        // 16-column blocks g, g + NG, ...; `add` = the slab already holds earlier flushes.
        auto flush = [&](bool add) {
            tc_fence_after();
            for (int cb = 16 * grp; cb < KP; cb += 16 * NG) {
                uint32_t a[16], bq[16];
                tmem_ld16(lane_base + T_ACC + cb, a);
                tmem_ld16(lane_base + T_ACC + KP + cb, bq);
                tmem_wait_ld();
                float4* sa = reinterpret_cast<float4*>(slab + (size_t)t * KP + cb);
                float4* sb = reinterpret_cast<float4*>(slab + (size_t)128 * KP + (size_t)t * KP + cb);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float4 va = make_float4(__uint_as_float(a[4 * j]), __uint_as_float(a[4 * j + 1]), __uint_as_float(a[4 * j + 2]), __uint_as_float(a[4 * j + 3]));
                    float4 vb = make_float4(__uint_as_float(bq[4 * j]), __uint_as_float(bq[4 * j + 1]), __uint_as_float(bq[4 * j + 2]), __uint_as_float(bq[4 * j + 3]));
                    if (add) {
                        const float4 oa = sa[j], ob = sb[j];
                        va.x += oa.x; va.y += oa.y; va.z += oa.z; va.w += oa.w;
                        vb.x += ob.x; vb.y += ob.y; vb.z += ob.z; vb.w += ob.w;
                    }
                    sa[j] = va; sb[j] = vb;
                }
            }
            tc_fence_before();
        };
        uint32_t sq = 0, it = 0;
        for (long long tile = blockIdx.x; tile < g.n_tiles; tile += gridDim.x, sq += slots_per_tile, ++it) {
            if (it > 0) wait(B_DONE);                    // every MMA of the previous tile is complete: Hs is free
            NMF_TRCW(TR_TILE, 0);
            if (it > 0 && it % FLUSH_TILES == 0) flush(it > FLUSH_TILES);    // (the MMA issuer restarts the accumulation
                                                         // with this tile; it waits for B_HS, which follows the flush)
            h0(sq);
            // ---- steps: chunk c = NG j + grp of super-chunk j lies in ring slot c / 2 (32 pixels); the slots of the other
            // groups are only observed (waited for and released), in ring order; thread = (frame 128 m + t, 16 pixels),
            // two halves of 8 ----
            bool pending = false;
            const int sw = t & 7;
            int sv = 0;                                  // X / Omega slots of this tile visited so far
            for (int j = 0; j < NSC2; ++j) {
                const int c = NG * j + grp;
                for (; sv < (c >> 1); ++sv) { wait_full(sq + NHS + sv); release(sq + NHS + sv); }
                const uint32_t seq = sq + NHS + (c >> 1);
                const unsigned char* xsl = wait_full(seq) + t * 128;     // X rows (128 bytes each, 128-byte swizzle) at +0, Omega rows at +16 KB
                sv = (c >> 1) + 1;
                NMF_TRCW(TR_FULL, c);
                wait(B_S0 + (j & 1)); tc_fence_after();
                NMF_TRCW(TR_S, c);
                const uint32_t zcol = lane_base + T_Z + 16 * NG * (j & 1) + 16 * grp;
                const uint32_t ecol = lane_base + T_E + 32 * grp;
                uint32_t s[16];
                if (active) { tmem_ld16(zcol, s); tmem_wait_ld(); }
                NMF_TRCW(TR_LD, c);
                if (pending) { wait(B_G0 + grp); tc_fence_after(); }      // this group's E columns are free again
                NMF_TRCW(TR_EFREE, c);
                if (active) {
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        float x[8], o[8];
#pragma unroll
                        for (int ch = 0; ch < 2; ++ch) {
                            float4 xv = make_float4(0.f, 0.f, 0.f, 0.f), ov = xv;
                            if (fr < N) {
                                const int cs = ((4 * (c & 1) + 2 * hf + ch) ^ sw) << 4;
                                xv = *reinterpret_cast<const float4*>(xsl + cs);
                                ov = *reinterpret_cast<const float4*>(xsl + 128 * PSW * 4 + cs);
                            }
                            x[4 * ch] = xv.x; x[4 * ch + 1] = xv.y; x[4 * ch + 2] = xv.z; x[4 * ch + 3] = xv.w;
                            o[4 * ch] = ov.x; o[4 * ch + 1] = ov.y; o[4 * ch + 2] = ov.z; o[4 * ch + 3] = ov.w;
                        }
                        Ew8 w;
                        ew8(x, o, &s[8 * hf], w);
                        ew8_store(zcol, ecol, hf, w);
                    }
                }
                release(seq);                            // after the values were consumed
                tmem_wait_st();
                tc_fence_before();
                warp_arrive(B_P0 + grp);
                NMF_TRCW(TR_HANDED, c);
                pending = true;
            }
            for (; sv < NSW; ++sv) { wait_full(sq + NHS + sv); release(sq + NHS + sv); }
            wait(B_G0 + grp);                            // this group's last AB of the tile is complete
        }
        wait(B_DONE);                                    // every MMA of the last tile is complete
        flush(it > FLUSH_TILES);                         // what was accumulated since the last flush (grid.x <= n_tiles:
                                                         // every CTA had a tile)
    }
    NMF_TRC_FLUSH(1);
    tc_fence_before();
    __syncthreads();
    if (warp == W_MMA) tmem_dealloc(tmem, 512);
}

// =====================================================================================================================
// W half-step (and projection), K <= 64: the same stages as k_tc_w, software-pipelined ACROSS tiles.
//
// In k_tc_w a tile is a closed sequence -- H pieces, S', element-wise chunks, AB -- and the tensor pipe idles while the
// next tile's H pieces are split and while the first chunks of a tile are computed (timeline: about 3 k of 9.5 k cycles
// per tile).  Here the H pieces are double-buffered (Hs[tile & 1]) and the MMA issuer runs one continuous stream
//     AB(t, chunks 0-3)  S'(t+1, 0)  AB(t, chunks 4-7)  S'(t+1, 1)  AB(t+1, chunks 0-3) ...
// while every element-wise group does   chunk(t, g)  H pieces (pixels 0-63) of t+1  chunk(t, 4 + g)  H pieces (64-127) ...
// The fp32 H' tile of tile t+1 does not pass through the ring: the TMA producer lands it, 64 pixels at a time, IN the
// buffer Hs[(t+1) & 1] as soon as the MMAs of tile t-1 that read those pixels are complete (B_DONE, B_DONEB) -- a whole
// tile before the pieces are needed; the element-wise warps read their values, meet at their group's named barrier and
// overwrite them with the pieces.  The ring (four 32 KB slots at K > 32) then holds X and Omega only: one
// full tile ahead.  The accumulators are flushed as in k_tc_w; around a flush the MMA issuer waits for the
// element-wise warps (B_FRDY / B_FDONE), S' of the next tile is still issued ahead.
// =====================================================================================================================
template <int KS>
__global__ void __launch_bounds__(32 * (4 * 4 + 2), 1)
k_tc_wp(const __grid_constant__ SplitArgs g) {
    constexpr int NG = 4;
    constexpr int KP = 16 * KS;
    constexpr int EW_WARPS = 4 * NG, W_MMA = EW_WARPS, W_TMA = EW_WARPS + 1;
    constexpr int NPT = npt_of(KP, NG, 2 * KP);
    static_assert(KS <= 4 && NPT == 3, "every piece of the M tile's rows of W lives in TMEM");
    constexpr uint32_t T_WT = 0;                                          // piece i at i KP / 2
    constexpr uint32_t T_Z = NPT * KP / 2, T_E = T_Z + 32 * NG;           // Z[jb] at T_Z + 16 NG jb, E[g] at T_E + 32 g
    constexpr uint32_t T_ACC = 512 - 2 * KP;                              // A at T_ACC, B at T_ACC + KP
    static_assert(T_E + 32 * NG <= T_ACC, "TMEM");
    constexpr int NBLK = KP / 16;
    constexpr int NSW = TILE / PSW;                      // X / Omega ring slots per tile
    constexpr int HS_BYTES = (KP / 8) * HS_SB;           // one BF16 piece of the H tile
    constexpr int HSBUF = 3 * HS_BYTES;                  // (the fp32 tile lands in the same buffer, see H0)
    extern __shared__ __align__(1024) unsigned char smem[];
    const int N = g.N, K = g.K;
    unsigned char* ring = smem;
    unsigned char* hs_p = ring + (size_t)g.NS * SLOTW;  // two buffers of 3 pieces of an H tile, [pixel][comp]
    uint64_t* bars = reinterpret_cast<uint64_t*>(hs_p + 2 * HSBUF);
    uint32_t* tptr = reinterpret_cast<uint32_t*>(bars + B_COUNT);
    const RingCtl rc{(uint32_t)g.NS, 0xffffffffu / (uint32_t)g.NS + 1u};

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int b = blockIdx.y, m = blockIdx.z;
    NMF_TRC_DECL;
    const float* __restrict__ W = g.W + (size_t)b * N * K;
    float* slab = g.slab + (((size_t)b * gridDim.z + m) * gridDim.x + blockIdx.x) * 2 * (size_t)128 * KP;
    // tiles of this CTA: blockIdx.x, blockIdx.x + gridDim.x, ...  (gridDim.x <= n_tiles: at least one)
    const uint32_t n_my = (uint32_t)((g.n_tiles - 1 - blockIdx.x) / gridDim.x) + 1u;

    if (tid == 0) {
        mbar_init(&bars[B_HS], EW_WARPS); mbar_init(&bars[B_HSB], EW_WARPS);
        for (int i = 0; i < 4; ++i) mbar_init(&bars[B_HFULL + i], 1);
        mbar_init(&bars[B_S0], 1); mbar_init(&bars[B_S1], 1); mbar_init(&bars[B_DONE], 1); mbar_init(&bars[B_DONEB], 1);
        mbar_init(&bars[B_FRDY], 1); mbar_init(&bars[B_FDONE], EW_WARPS);
        for (int i = 0; i < NG; ++i) { mbar_init(&bars[B_P0 + i], 4); mbar_init(&bars[B_G0 + i], 1); }
        // every element-wise warp waits for and releases EVERY ring slot (see "Ring slots and groups")
        for (int s = 0; s < g.NS; ++s) { mbar_init(&bars[B_FULL + s], 1); mbar_init(&bars[B_EMPTY + s], EW_WARPS); }
        mbar_fence_init();
    }
    if (warp == W_MMA) tmem_alloc(tptr, 512);
    if (warp == W_TMA && lane == 0) { tma_prefetch_desc(&g.mH); tma_prefetch_desc(&g.mX); tma_prefetch_desc(&g.mO); }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tptr;
    const uint32_t hs_s = smem_u32(hs_p), ring_s = smem_u32(ring);

    if (warp < EW_WARPS) {
        // the M tile's rows of W -> TMEM (A operand of S', fixed for the launch); lane = frame 128 m + t
        const int q = warp & 3, grp = warp >> 2, t = 32 * q + lane;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const int fr = 128 * m + t;
        for (int bi = grp; bi < NBLK; bi += NG) {
            uint32_t p[3][8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int k0 = 16 * bi + 2 * j;
                const float w0 = (fr < N && k0 < K) ? W[(size_t)fr * K + k0] : 0.f;
                const float w1 = (fr < N && k0 + 1 < K) ? W[(size_t)fr * K + k0 + 1] : 0.f;
                split3_pair(w0, w1, p[0][j], p[1][j], p[2][j]);
            }
#pragma unroll
            for (int i = 0; i < 3; ++i) tmem_st8(lane_base + T_WT + i * (KP / 2) + 8 * bi, p[i]);
        }
        tmem_wait_st();
        tc_fence_before();
    }
    __syncthreads();
    tc_fence_after();

    if (warp == W_TMA) {
        // =========================== TMA producer ===========================
        // Per tile i, in the order in which they become possible: X / Omega slots 0, 1 of the tile; the first 64 pixels of
        // the fp32 H' tile of tile i + 1 into Hs[(i + 1) & 1] (those rows are free once AB of chunks 0-3 of tile i - 1 is
        // complete, B_DONE); slots 2, 3; the other 64 pixels (free after chunks 4-7 of tile i - 1, B_DONEB).
        if (lane == 0) {
            uint32_t seq = 0, ph_a = 0, ph_b = 0;
            auto acquire = [&](uint32_t bytes) -> uint32_t {
                uint32_t par;
                const uint32_t s = rc.slot(seq, par);
                mbar_wait(&bars[B_EMPTY + s], par ^ 1u);
                mbar_expect_tx(&bars[B_FULL + s], bytes);
                ++seq;
                return s;
            };
            // half hf of the H' tile of tile i: rows 16 g + 4 r .. + 3 ([4 comps][64 px] = 1 KB) land where group g writes
            // its part of piece r / 2 (see H0)
            auto load_h = [&](uint32_t i, uint32_t hf) {
                const int p0 = (int)((blockIdx.x + (long long)i * gridDim.x) * TILE) + 64 * (int)hf;
                uint64_t* bar = &bars[B_HFULL + 2 * (i & 1u) + hf];
                const uint32_t dst = hs_s + (i & 1u) * HSBUF + 1024 * hf;
                mbar_expect_tx(bar, NBLK * 16 * 64 * 4);
                for (int gb = 0; gb < NBLK; ++gb)
#pragma unroll
                    for (int r = 0; r < 4; ++r)
                        tma_load_2d(dst + (r >> 1) * HS_BYTES + (2 * gb + (r & 1)) * HS_SB, &g.mH, p0, b * K + 16 * gb + 4 * r, bar);
            };
            auto load_x = [&](uint32_t i, int c) {
                const int p0 = (int)((blockIdx.x + (long long)i * gridDim.x) * TILE);
                const uint32_t s = acquire(SLOTW);
                NMF_TRCW(TR_T_ACQ, 1 + c);
                tma_load_2d(ring_s + s * SLOTW, &g.mX, p0 + PSW * c, b * N + 128 * m, &bars[B_FULL + s]);
                tma_load_2d(ring_s + s * SLOTW + 128 * PSW * 4, &g.mO, p0 + PSW * c, b * N + 128 * m, &bars[B_FULL + s]);
            };
            load_h(0, 0); load_h(0, 1);
            for (uint32_t i = 0; i < n_my; ++i) {
                load_x(i, 0); load_x(i, 1);
                if (i + 1 < n_my) {
                    if (i >= 1) { mbar_wait(&bars[B_DONE], ph_a); ph_a ^= 1u; }        // chunks 0-3 of tile i - 1 are complete
                    NMF_TRCW(TR_T_ACQ, 0);
                    load_h(i + 1, 0);
                }
                load_x(i, 2); load_x(i, 3);
                if (i + 1 < n_my) {
                    if (i >= 1) { mbar_wait(&bars[B_DONEB], ph_b); ph_b ^= 1u; }       // chunks 4-7 of tile i - 1 are complete
                    load_h(i + 1, 1);
                }
            }
        }
    } else if (warp == W_MMA) {
        // =========================== MMA issuer ===========================
        uint32_t ph = 0;
        auto wait = [&](int bar) { mbar_wait(&bars[bar], (ph >> bar) & 1u); ph ^= 1u << bar; tc_fence_after(); };
        constexpr uint32_t id_s = idesc_bf16(128, 16 * NG, 0), id_ab = idesc_bf16(128, KP, 1);
        uint64_t d_hs_k[3], d_hs_mn[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            d_hs_k[i] = smem_desc(hs_s + i * HS_BYTES, HS_SB, 128);
            d_hs_mn[i] = smem_desc(hs_s + i * HS_BYTES, 128, HS_SB);
        }
        constexpr uint32_t hs_kstep = (uint32_t)(2 * HS_SB) >> 4;
        constexpr uint32_t hs_buf = (uint32_t)HSBUF >> 4;
        auto issue_S2 = [&](uint32_t hb, int j) {        // S'(j): [128 frames] x [64 px], K = comps, from Hs[hb] -> Z[j]
            if (elect_one()) {
                const uint32_t boff = hb * hs_buf + ((uint32_t)(j * NG * 2 * 128) >> 4);
                const uint32_t d = tmem + T_Z + 16 * NG * j;
#pragma unroll
                for (int pr = 0; pr < 6; ++pr)
#pragma unroll
                    for (int ks = 0; ks < KS; ++ks)
                        mma16_ts(d, tmem + T_WT + PA[pr] * (KP / 2) + 8 * ks, d_hs_k[PB[pr]] + boff + ks * hs_kstep, id_s,
                                 (pr | ks) ? 1u : 0u);
                mma_commit(&bars[B_S0 + j]);
            }
            __syncwarp();
        };
        bool acc_started = false;
        wait(B_HS);
        NMF_TRCW(TR_M_HS, 0);
        issue_S2(0, 0);
        wait(B_HSB);
        issue_S2(0, 1);
        NMF_TRCW(TR_M_S, 1);
        for (uint32_t it = 0; it < n_my; ++it) {
            const uint32_t hb = it & 1u;
            if (it % FLUSH_TILES == 0) {
                acc_started = false;                     // the accumulators were flushed into the slab
                if (it > 0) wait(B_FDONE);
            }
            for (int j = 0; j < 2; ++j) {
                for (int gg = 0; gg < NG; ++gg) {
                    const int c = NG * j + gg;
                    wait(B_P0 + gg);
                    NMF_TRCW(TR_M_READY, c);
                    if (elect_one()) {
                        const uint32_t boff = hb * hs_buf + ((uint32_t)(c * 2 * 128) >> 4);   // 16 pixels = 2 row groups
                        const uint32_t z = tmem + T_Z + 16 * NG * j + 16 * gg, e = tmem + T_E + 32 * gg;
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
                    NMF_TRCW(TR_M_ISSUED, c);
                    acc_started = true;
                }
                if (elect_one()) mma_commit(&bars[j ? B_DONEB : B_DONE]);   // pixels 64 j .. + 63 of Hs[hb] may be rewritten
                __syncwarp();
                if (it + 1 < n_my) {                     // the next tile's S'(j): Z[j] is free, its R pieces were read by
                    wait(j ? B_HSB : B_HS);              // the MMAs just issued (the pipe is in order)
                    NMF_TRCW(TR_M_HS, j);
                    issue_S2(hb ^ 1u, j);
                    NMF_TRCW(TR_M_S, j);
                }
            }
            if ((it + 1) % FLUSH_TILES == 0 || it + 1 == n_my) {
                if (elect_one()) mma_commit(&bars[B_FRDY]);
                __syncwarp();
            }
        }
    } else if (warp < EW_WARPS) {
        // =========================== element-wise warps: group grp = warp / 4, lane quadrant q = warp % 4 ===========================
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
        // H0, one half (64 pixels) of a tile at a time: the fp32 values of the H' tile that landed in Hs[hb] are replaced
        // by the pieces Hs[hb][pixel][comp].  Group g takes the 16-component block g; thread = (pixel 64 hf + t % 64,
        // components 8 (t / 64) .. + 7 of the block).  The fp32 rows of the block (four boxes of [4 comps][64 px], 1 KB
        // each) lie exactly where group g writes its part of pieces 0 and 1, so a group only ever overwrites what its
        // own threads have read: they read, meet at the group's named barrier, and write.
        auto h0 = [&](uint32_t hb, uint32_t hf) {
            NMF_TRCW(TR_H0_BEGIN, hf);
            wait(B_HFULL + 2 * (int)hb + (int)hf);
            NMF_TRCW(TR_HSLOT, hf);
            if (grp < NBLK) {
                const int kh = q >> 1, px = t & 63, kg = 2 * grp + kh;
                unsigned char* buf = hs_p + (size_t)hb * HSBUF;
                const unsigned char* land = buf + kh * HS_BYTES + 2 * grp * HS_SB + 1024 * hf + 4 * px;   // boxes r = 2 kh, 2 kh + 1
                float h[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) h[j] = *reinterpret_cast<const float*>(land + (j >> 2) * HS_SB + (j & 3) * 256);
                if (8 * kg + 8 > K) {                    // rows at or beyond K hold another problem's data or zeros
#pragma unroll
                    for (int j = 0; j < 8; ++j) if (8 * kg + j >= K) h[j] = 0.f;
                }
                uint32_t p[3][4];
#pragma unroll
                for (int j = 0; j < 4; ++j) split3_pair(h[2 * j], h[2 * j + 1], p[0][j], p[1][j], p[2][j]);
                asm volatile("bar.sync %0, 128;" ::"r"(1 + grp) : "memory");
#pragma unroll
                for (int i = 0; i < 3; ++i) st_piece_smem(buf + i * HS_BYTES, 64 * (int)hf + px, kg, p[i]);
                fence_proxy_async();
            }
            warp_arrive(hf ? B_HSB : B_HS);
            NMF_TRCW(TR_H0_END, hf);
        };
        auto flush = [&](bool add) {                     // see k_tc_w
            tc_fence_after();
            for (int cb = 16 * grp; cb < KP; cb += 16 * NG) {
                uint32_t a[16], bq[16];
                tmem_ld16(lane_base + T_ACC + cb, a);
                tmem_ld16(lane_base + T_ACC + KP + cb, bq);
                tmem_wait_ld();
                float4* sa = reinterpret_cast<float4*>(slab + (size_t)t * KP + cb);
                float4* sb = reinterpret_cast<float4*>(slab + (size_t)128 * KP + (size_t)t * KP + cb);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float4 va = make_float4(__uint_as_float(a[4 * j]), __uint_as_float(a[4 * j + 1]), __uint_as_float(a[4 * j + 2]), __uint_as_float(a[4 * j + 3]));
                    float4 vb = make_float4(__uint_as_float(bq[4 * j]), __uint_as_float(bq[4 * j + 1]), __uint_as_float(bq[4 * j + 2]), __uint_as_float(bq[4 * j + 3]));
                    if (add) {
                        const float4 oa = sa[j], ob = sb[j];
                        va.x += oa.x; va.y += oa.y; va.z += oa.z; va.w += oa.w;
                        vb.x += ob.x; vb.y += ob.y; vb.z += ob.z; vb.w += ob.w;
                    }
                    sa[j] = va; sb[j] = vb;
                }
            }
            tc_fence_before();
        };
        h0(0, 0); h0(0, 1);
        uint32_t sq = 0;
        bool pending = false;
        const int sw = t & 7;
        for (uint32_t it = 0; it < n_my; ++it, sq += NSW) {
            if (it > 0 && it % FLUSH_TILES == 0) {
                wait(B_FRDY); flush(it > FLUSH_TILES);   // every MMA up to the previous tile is complete; the MMA issuer
                warp_arrive(B_FDONE);                    // restarts the accumulation once every warp has flushed
            }
            // chunk c = NG j + grp lies in ring slot c / 2 (32 pixels); the slots of the other groups are only observed
            // (waited for and released), in ring order; thread = (frame 128 m + t, 16 pixels), two halves of 8
            int sv = 0;
            for (int j = 0; j < 2; ++j) {
                const int c = NG * j + grp;
                for (; sv < (c >> 1); ++sv) { wait_full(sq + sv); release(sq + sv); }
                const uint32_t seq = sq + (c >> 1);
                const unsigned char* xsl = wait_full(seq) + t * 128;     // X rows (128 bytes each, 128-byte swizzle) at +0, Omega rows at +16 KB
                sv = (c >> 1) + 1;
                NMF_TRCW(TR_FULL, c);
                wait(B_S0 + j); tc_fence_after();
                NMF_TRCW(TR_S, c);
                const uint32_t zcol = lane_base + T_Z + 16 * NG * j + 16 * grp;
                const uint32_t ecol = lane_base + T_E + 32 * grp;
                uint32_t s[16];
                if (active) { tmem_ld16(zcol, s); tmem_wait_ld(); }
                NMF_TRCW(TR_LD, c);
                if (pending) { wait(B_G0 + grp); tc_fence_after(); }      // this group's E columns are free again
                NMF_TRCW(TR_EFREE, c);
                if (active) {
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        float x[8], o[8];
#pragma unroll
                        for (int ch = 0; ch < 2; ++ch) {
                            float4 xv = make_float4(0.f, 0.f, 0.f, 0.f), ov = xv;
                            if (fr < N) {
                                const int cs = ((4 * (c & 1) + 2 * hf + ch) ^ sw) << 4;
                                xv = *reinterpret_cast<const float4*>(xsl + cs);
                                ov = *reinterpret_cast<const float4*>(xsl + 128 * PSW * 4 + cs);
                            }
                            x[4 * ch] = xv.x; x[4 * ch + 1] = xv.y; x[4 * ch + 2] = xv.z; x[4 * ch + 3] = xv.w;
                            o[4 * ch] = ov.x; o[4 * ch + 1] = ov.y; o[4 * ch + 2] = ov.z; o[4 * ch + 3] = ov.w;
                        }
                        Ew8 w;
                        ew8(x, o, &s[8 * hf], w);
                        ew8_store(zcol, ecol, hf, w);
                    }
                }
                release(seq);                            // after the values were consumed
                tmem_wait_st();
                tc_fence_before();
                warp_arrive(B_P0 + grp);
                NMF_TRCW(TR_HANDED, c);
                pending = true;
                if (it + 1 < n_my) h0((it + 1) & 1u, (uint32_t)j);       // the next tile's H pieces, half j
            }
            for (; sv < NSW; ++sv) { wait_full(sq + sv); release(sq + sv); }
        }
        if (pending) wait(B_G0 + grp);
        wait(B_FRDY);                                    // every MMA of the launch is complete
        flush(n_my > FLUSH_TILES);
    }
    NMF_TRC_FLUSH(1);
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
// groups of element-wise warps: four chunks in flight where at least two pieces of the TMEM-resident operand still fit
inline int ng_of(int KP) { return KP <= 80 ? 4 : 2; }
inline size_t smem_fixed_h(int NF, int KP, int NG) {
    return (size_t)3 * KP * NF * 2 + (size_t)(3 - npt_of(KP, NG, 2 * KP)) * (KP / 8) * HS_SB + B_COUNT * 8 + 16;
}
inline size_t smem_fixed_w(int KP, int NG) {
    return (size_t)(3 + 3 - npt_of(KP, NG, 2 * KP)) * (KP / 8) * HS_SB + B_COUNT * 8 + 16;
}
inline size_t smem_fixed_wp(int KP) { return (size_t)2 * 3 * (KP / 8) * HS_SB + B_COUNT * 8 + 16; }
// Which W kernel: the pipelined one (k_tc_wp, K <= 64) wins where the element-wise load per tile is light -- the
// projection of up to 64 frames (at most two of the four lane quadrants hold frames): 0.226 ms against 0.283 ms for 32
// frames at 1024^2, K = 50.  With all 128 lanes busy (the fit) its MMAs and the element-wise warps run at the same time
// and slow each other down -- 30 % more tensor-active cycles for the same MMAs -- and it is 5 % SLOWER than k_tc_w
// (DESIGN.md 6.2), so the fit keeps k_tc_w.
inline bool use_wp(int KP, bool fit, int rows) { return KP <= 64 && !fit && rows <= 64; }
// ring slots that fit beside `fixed` bytes, rounded down to a multiple of `mult` (see "Ring slots and groups")
inline int slots_for(size_t fixed, int slot_bytes, int mult) {
    long long ns = ((long long)SMEM_MAX - (long long)fixed) / slot_bytes;
    if (ns > MAX_SLOTS) ns = MAX_SLOTS;
    return ns < 0 ? 0 : (int)(ns / mult * mult);
}
// the opt-in shared-memory size is a per-device function attribute: set once per device and instantiation
template <typename Kern>
cudaError_t set_smem_attr_once(Kern kern, bool (&done)[NMF_MAX_DEVICES], int device) {
    if (device >= 0 && device < NMF_MAX_DEVICES && done[device]) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
    if (e == cudaSuccess && device >= 0 && device < NMF_MAX_DEVICES) done[device] = true;
    return e;
}
template <int KS, int NG>
cudaError_t launch_h(const SplitArgs& a, dim3 grid, size_t smem, cudaStream_t st, int device) {
    static bool done[NMF_MAX_DEVICES] = {};
    cudaError_t e = set_smem_attr_once(k_tc_h<KS, NG>, done, device);
    if (e != cudaSuccess) return e;
    k_tc_h<KS, NG><<<grid, 32 * (4 * NG + 2), smem, st>>>(a);
    return cudaSuccess;
}
template <int KS, int NG>
cudaError_t launch_w(const SplitArgs& a, dim3 grid, size_t smem, cudaStream_t st, int device) {
    static bool done[NMF_MAX_DEVICES] = {};
    cudaError_t e = set_smem_attr_once(k_tc_w<KS, NG>, done, device);
    if (e != cudaSuccess) return e;
    k_tc_w<KS, NG><<<grid, 32 * (4 * NG + 2), smem, st>>>(a);
    return cudaSuccess;
}
template <int KS>
cudaError_t launch_wp(const SplitArgs& a, dim3 grid, size_t smem, cudaStream_t st, int device) {
    static bool done[NMF_MAX_DEVICES] = {};
    cudaError_t e = set_smem_attr_once(k_tc_wp<KS>, done, device);
    if (e != cudaSuccess) return e;
    k_tc_wp<KS><<<grid, 32 * (4 * 4 + 2), smem, st>>>(a);
    return cudaSuccess;
}
inline cudaError_t launch_wp_ks(int KS, const SplitArgs& a, dim3 grid, size_t smem, cudaStream_t st, int device) {
    return KS == 1 ? launch_wp<1>(a, grid, smem, st, device) : KS == 2 ? launch_wp<2>(a, grid, smem, st, device) :
           KS == 3 ? launch_wp<3>(a, grid, smem, st, device) : launch_wp<4>(a, grid, smem, st, device);
}
// KS = 1 .. 5 (KP <= 80) run with four groups, KS = 6 .. 8 with two (ng_of)
#define NMF_KS_SWITCH(fn, KS, ...)                                    \
    ((KS) == 1 ? fn<1, 4>(__VA_ARGS__) : (KS) == 2 ? fn<2, 4>(__VA_ARGS__) : (KS) == 3 ? fn<3, 4>(__VA_ARGS__) : \
     (KS) == 4 ? fn<4, 4>(__VA_ARGS__) : (KS) == 5 ? fn<5, 4>(__VA_ARGS__) : (KS) == 6 ? fn<6, 2>(__VA_ARGS__) : \
     (KS) == 7 ? fn<7, 2>(__VA_ARGS__) : fn<8, 2>(__VA_ARGS__))

// persistent CTAs for `n_tiles` tiles on `avail` SMs, evened out so that every CTA gets `per` or `per - 1` tiles
inline int even_ctas(long long n_tiles, long long avail) {
    if (avail < 1) avail = 1;
    if (avail > n_tiles) avail = n_tiles;
    const long long per = (n_tiles + avail - 1) / avail;
    return (int)((n_tiles + per - 1) / per);
}

// iters x { W half-step (+ optionally the H half-step before it) ; reduce + update }
int split_run(nmf_plan* p, const float* X, const float* Om, float* W, float* H, int rows, int iters, int batch, bool fit) {
    const int KP = kp_of(p->K), KS = KP / 16, NG = ng_of(KP);
    const int MT = (rows + 127) / 128;
    const long long n_tiles = (p->P + TILE - 1) / TILE;
    const long long trows = (long long)batch * rows;
    SplitArgs h{}, w{};
    h.W = w.W = W; h.H = w.H = H; w.slab = h.slab = reinterpret_cast<float*>(p->ws);
    h.N = w.N = rows; h.K = w.K = p->K; h.P = w.P = p->P; h.n_tiles = w.n_tiles = n_tiles;
    h.NF = w.NF = (rows + FCH - 1) / FCH * FCH; h.NC = w.NC = h.NF / FCH;
    const bool wp = use_wp(KP, fit, rows) && slots_for(smem_fixed_wp(KP), SLOTW, 1) >= 2;
    const size_t fixed_w = wp ? smem_fixed_wp(KP) : smem_fixed_w(KP, NG);
    h.NS = slots_for(smem_fixed_h(h.NF, KP, NG), SLOT, NG); w.NS = slots_for(fixed_w, SLOTW, 1);
    bool ok = make_map(&w.mH, H, (long long)batch * p->K, p->P, wp ? 4 : 64, wp ? 64 : TILE, 0) &&
              make_map(&w.mX, X, trows, p->P, 128, PSW, 128) && make_map(&w.mO, Om, trows, p->P, 128, PSW, 128);
    if (fit) ok = ok && make_map(&h.mH, H, (long long)batch * p->K, p->P, 16, TILE, 0) &&
                  make_map(&h.mX, X, trows, p->P, FCH, TILE, 0) && make_map(&h.mO, Om, trows, p->P, FCH, TILE, 0);
    if (!ok) {
        if (!p->sticky) { p->sticky = NMF_ERR_CUDA; p->cuda_msg = "cuTensorMapEncodeTiled failed"; }
        return NMF_ERR_CUDA;
    }
    const int ctas_h = even_ctas(n_tiles, p->num_sms / batch);
    const int ctas_w = even_ctas(n_tiles, p->num_sms / (batch * MT));
    const size_t smem_h = smem_fixed_h(h.NF, KP, NG) + (size_t)h.NS * SLOT;
    const size_t smem_w = fixed_w + (size_t)w.NS * SLOTW;
    const int nk = rows * p->K;
    int rc = nmf_run_iterations(p, fit ? 40 : 41, X, Om, W, H, nullptr, rows, batch, iters, [&]() -> int {
        if (fit) {
            NMF_CUDA_TRY(p, NMF_KS_SWITCH(launch_h, KS, h, dim3(ctas_h, batch), smem_h, p->stream, p->device));
            p->launches++;
        }
        if (wp) NMF_CUDA_TRY(p, launch_wp_ks(KS, w, dim3(ctas_w, batch, MT), smem_w, p->stream, p->device));
        else NMF_CUDA_TRY(p, NMF_KS_SWITCH(launch_w, KS, w, dim3(ctas_w, batch, MT), smem_w, p->stream, p->device));
        k_w_update_split<<<dim3((nk + WU_E - 1) / WU_E, batch), WU_E * WU_Q, 0, p->stream>>>(w.slab, W, rows, p->K, KP, ctas_w, MT);
        p->launches += 2;
        return NMF_OK;
    });
    if (rc) return rc;
    NMF_CUDA_TRY(p, cudaGetLastError());
    return NMF_OK;
}

}  // namespace

void nmf_tcsplit_configure(nmf_plan* p) {
    p->s_ok = false;
    if (p->K > 128 || p->N > 256) return;
    if (p->P + TILE >= (1LL << 31) || (long long)p->batch * p->N >= (1LL << 31)) return;   // TMA coordinates are int32
    const int KP = kp_of(p->K), NG = ng_of(KP), NF = (p->N + FCH - 1) / FCH * FCH;
    if (slots_for(smem_fixed_h(NF, KP, NG), SLOT, NG) < NG ||
        slots_for(smem_fixed_w(KP, NG), SLOTW, 1) < 2) return;
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

#ifdef NMF_TC_TRACE
// trace build only (build.py build_trace): copies the event log of CTA (0, 0, 0) of the last split-kernel launches:
// counts[2][18] events per kernel (k_tc_h, k_tc_w) and warp, events[2][18][2048] = event << 56 | argument << 48 | clock64
extern "C" int nmf_debug_trace(unsigned int* counts_host, unsigned long long* events_host, int reset) {
    if (cudaMemcpyFromSymbol(counts_host, tc::g_trace_n, sizeof(unsigned int) * tc::TRACE_KERNELS * tc::TRACE_WARPS) != cudaSuccess) return -1;
    if (cudaMemcpyFromSymbol(events_host, tc::g_trace, sizeof(unsigned long long) * tc::TRACE_KERNELS * tc::TRACE_WARPS * tc::TRACE_LEN) != cudaSuccess) return -1;
    if (reset) {
        unsigned int z[tc::TRACE_KERNELS * tc::TRACE_WARPS] = {};
        if (cudaMemcpyToSymbol(tc::g_trace_n, z, sizeof(z)) != cudaSuccess) return -1;
    }
    return tc::TRACE_LEN;
}
#endif

#ifdef NMF_WAIT_DEBUG
// debugging build only: copies the wait log of this translation unit (entries of 4 words) to `out_host`
extern "C" int nmf_debug_wait_log(unsigned int* out_host, int max_entries) {
    unsigned int n = 0;
    if (cudaMemcpyFromSymbol(&n, tc::g_wait_log_n, sizeof(n)) != cudaSuccess) return -1;
    if ((int)n > max_entries) n = max_entries;
    if (n > 256) n = 256;
    if (n && cudaMemcpyFromSymbol(out_host, tc::g_wait_log, n * 4 * sizeof(unsigned int)) != cudaSuccess) return -1;
    return (int)n;
}
#endif

// nmf_tc.cuh -- sm_100a primitives used by the tensor-core NMF kernel (inline PTX only):
// mbarrier, TMA (cp.async.bulk.tensor), proxy/tcgen05 fences, TMEM allocation, tcgen05.ld/st, the UMMA
// shared-memory descriptor and tcgen05.commit.  (The kind::f16 MMA wrappers live next to the kernel.)
//
// Operand layout (no-swizzle canonical form, 16-bit elements, 8 per 16 bytes):
//   a buffer Z[a][b] is stored as 8x8 core matrices (8 consecutive a, 8 consecutive b, 128 bytes):
//       byte(a, b) = (a % 8) * 16 + (a / 8) * 128 + (b % 8) * 2 + (b / 8) * SB
//   * read as a K-major operand   (MN = a, K = b): SBO = 128, LBO = SB, one MMA (K = 16) spans 2 LBO
//   * read as an MN-major operand (MN = b, K = a): SBO = SB, LBO = 128, one MMA (K = 16) spans 2 row groups
// so the same bytes serve W (frames x components) and H^T (pixels x components) in both roles.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tc {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---------------------------------------------------------------- mbarrier
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// try_wait with a suspend-time hint: the warp sleeps in hardware for up to `ns` and is woken by the completing
// arrive, instead of re-issuing the probe every few tens of cycles (a spinning warp takes issue slots from the
// compute warps that share its scheduler).
__device__ __forceinline__ bool mbar_try_wait_hint(uint64_t* bar, uint32_t parity, uint32_t ns) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug traps (launch error surfaced by the C-ABI) instead of hanging the GPU.  Each failed
// probe has already slept in hardware for the try_wait time limit, so the loop is two instructions per wake-up (the
// suspend-time-hint form compiles to TRYWAIT + NANOSLEEP.SYNCS + a second probe and woke about twenty times per
// wait: a third of all instructions the element-wise warps issued); 2^26 failed probes are far beyond any legitimate
// wait (a whole launch takes milliseconds).
#ifdef NMF_WAIT_DEBUG
// debugging build (python -m paper_2309_04623_b200.build --wait-debug): a wait that times out is recorded (block, warp,
// shared-memory address of the barrier, parity) and abandoned instead of trapping, so the log survives the launch
__device__ unsigned int g_wait_log[4 * 256];
__device__ unsigned int g_wait_log_n;
#endif
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t n = 0;
    while (!mbar_try_wait(bar, parity)) {
#ifdef NMF_WAIT_DEBUG
        if (++n > (1u << 22)) {
            if ((threadIdx.x & 31) == 0 || true) {
                const unsigned int i = atomicAdd(&g_wait_log_n, 1u);
                if (i < 256) {
                    g_wait_log[4 * i] = blockIdx.x | (blockIdx.y << 12) | (blockIdx.z << 24);
                    g_wait_log[4 * i + 1] = threadIdx.x;
                    g_wait_log[4 * i + 2] = smem_u32(bar);
                    g_wait_log[4 * i + 3] = parity;
                }
            }
            return;
        }
#else
        if (++n > (1u << 26)) __trap();
#endif
    }
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

// ---------------------------------------------------------------- timeline trace (python bench.py --trace)
// With -DNMF_TC_TRACE (build.py build_trace) lane 0 of every warp of CTA (0, 0, 0) records (event, argument, clock64)
// at the hand-over points of the split kernels; nmf_debug_trace copies the log out.  Compiled out of the product.
#ifdef NMF_TC_TRACE
constexpr int TRACE_WARPS = 18, TRACE_LEN = 2048, TRACE_KERNELS = 2;
__device__ unsigned long long g_trace[TRACE_KERNELS * TRACE_WARPS * TRACE_LEN];
__device__ unsigned int g_trace_n[TRACE_KERNELS * TRACE_WARPS];
// the event counter lives in a register of the recording lane (a counter in global memory cost a round trip per event)
__device__ __forceinline__ void trace_event(int kern, int warp, int lane, unsigned& n, unsigned ev, unsigned arg) {
    if (lane == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && n < TRACE_LEN) {
        g_trace[(kern * TRACE_WARPS + warp) * TRACE_LEN + n] =
            ((unsigned long long)ev << 56) | ((unsigned long long)(arg & 0xffu) << 48) | ((unsigned long long)clock64() & 0xffffffffffffULL);
        ++n;
    }
}
__device__ __forceinline__ void trace_flush(int kern, int warp, int lane, unsigned n) {
    if (lane == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) g_trace_n[kern * TRACE_WARPS + warp] = n;
}
#define NMF_TRC_DECL unsigned trc_n = 0
#define NMF_TRC(ev, arg) tc::trace_event(0, warp, lane, trc_n, (ev), (arg))
#define NMF_TRCW(ev, arg) tc::trace_event(1, warp, lane, trc_n, (ev), (arg))
#define NMF_TRC_FLUSH(kern) tc::trace_flush((kern), warp, lane, trc_n)
#else
#define NMF_TRC_DECL do { } while (0)
#define NMF_TRC(ev, arg) do { } while (0)
#define NMF_TRCW(ev, arg) do { } while (0)
#define NMF_TRC_FLUSH(kern) do { } while (0)
#endif
// trace events: element-wise warps 1 slot landed, 2 S ready, 3 S loaded, 4 piece columns free, 5 pieces stored + chunk
// handed over, 6 H pieces begin, 7 H pieces done, 8 update begin, 9 update done; MMA issuer 16 pieces of a chunk ready,
// 17 its MMAs issued, 18 S series issued, 19 H pieces ready; k_tc_w only: 10 previous tile's MMAs complete, 11 H slot
// landed; TMA producer 24 ring slot acquired (argument = item of the tile)
enum { TR_FULL = 1, TR_S, TR_LD, TR_EFREE, TR_HANDED, TR_H0_BEGIN, TR_H0_END, TR_UPD_BEGIN, TR_UPD_END, TR_TILE, TR_HSLOT,
       TR_M_READY = 16, TR_M_ISSUED, TR_M_S, TR_M_HS, TR_T_ACQ = 24 };

// ---------------------------------------------------------------- TMA (cp.async.bulk.tensor, 2-D tiled maps)
// Loads the box of `tmap` whose first element is (x = innermost coordinate, y = row) into shared memory at
// `smem_dst`; the bytes (out-of-range elements arrive as zeros and are counted) complete on `bar`.
__device__ __forceinline__ void tma_load_2d(uint32_t smem_dst, const void* tmap, int x, int y, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(smem_dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(x), "r"(y), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const void* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tmap)) : "memory");
}

// ---------------------------------------------------------------- fences
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---------------------------------------------------------------- TMEM allocation (one full warp)
__device__ __forceinline__ void tmem_alloc(uint32_t* smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_dst)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}

// ---------------------------------------------------------------- TMEM <-> registers (lane = thread of the warp's quadrant)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t (&r)[4]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// ---------------------------------------------------------------- descriptors
// shared-memory matrix descriptor, no swizzle; byte offsets must be multiples of 16
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// all previously issued MMAs of this thread arrive on `bar` when complete (implies fence::before_thread_sync)
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------- kind::f16 MMA (BF16 operands, FP32 accumulation)
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

// exact 3-way BF16 split of two FP32 values, packed (low half = first value): x = x1 + x2 + x3 with
// x1 = x rounded to 8 significant bits (half away from zero), x2 = the next 8 bits of the remainder (truncated),
// x3 = what is left (at most 8 significant bits, so it is a BF16 number).  Integer / FADD / PRMT only: the
// F2FP conversion pipe is a quarter-rate unit and was the limiter of the element-wise warps in round 1 (in round 2, with
// 16 element-wise warps, piece 1 by one packed cvt.rn.bf16x2.f32 per pair -- two integer instructions fewer -- measured
// the same as this form: the split arithmetic is not what bounds the kernels).
__device__ __forceinline__ void split3_pair(float x0, float x1, uint32_t& p1, uint32_t& p2, uint32_t& p3) {
    const uint32_t a0 = (__float_as_uint(x0) + 0x8000u) & 0xffff0000u;
    const uint32_t a1 = (__float_as_uint(x1) + 0x8000u) & 0xffff0000u;
    p1 = __byte_perm(a0, a1, 0x7632);
    const float r0 = x0 - __uint_as_float(a0);
    const float r1 = x1 - __uint_as_float(a1);
    const uint32_t b0 = __float_as_uint(r0) & 0xffff0000u;
    const uint32_t b1 = __float_as_uint(r1) & 0xffff0000u;
    const float s0 = r0 - __uint_as_float(b0);
    const float s1 = r1 - __uint_as_float(b1);
    p2 = __byte_perm(b0, b1, 0x7632);
    p3 = __byte_perm(__float_as_uint(s0), __float_as_uint(s1), 0x7632);
}

__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
          "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
          "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}


// ---------------------------------------------------------------- element-wise stage shared by the tensor-core kernels
// layout of a group's E buffer (32 TMEM columns): R3, Q1, Q2, Q3, 8 columns (16 BF16 values) each
constexpr uint32_t O_R3 = 0, O_Q1 = 8, O_Q2 = 16, O_Q3 = 24;
// q = Om*X, r = Om*S for 16 consecutive elements (Omega == 0: missing datum, skipped (G5); X may be NaN/Inf
// there), split into BF16 pieces.  R1, R2 go back over S in place (`zcol`, this thread's lane); R3 and the Q pieces
// are returned packed in `e` for the single-buffered E columns.
__device__ __forceinline__ void ew16(const float (&x)[16], const float (&o)[16], const uint32_t (&s)[16], uint32_t zcol,
                                     uint32_t (&e)[32]) {
    uint32_t R1[8], R2[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float o0 = o[2 * i], o1 = o[2 * i + 1];
        const float q0 = o0 > 0.f ? o0 * x[2 * i] : 0.f;
        const float q1 = o1 > 0.f ? o1 * x[2 * i + 1] : 0.f;
        const float r0 = o0 * __uint_as_float(s[2 * i]);          // S is finite: Omega == 0 gives exactly 0
        const float r1 = o1 * __uint_as_float(s[2 * i + 1]);
        split3_pair(q0, q1, e[O_Q1 + i], e[O_Q2 + i], e[O_Q3 + i]);
        split3_pair(r0, r1, R1[i], R2[i], e[O_R3 + i]);
    }
    tmem_st8(zcol, R1); tmem_st8(zcol + 8, R2);
}

// The same stage for 8 consecutive elements (half a chunk), for the kernels that keep more chunks in flight with
// fewer registers per thread: every piece comes back as 4 words (columns 4 h .. 4 h + 3 of its 8-column block for
// half h).
struct Ew8 { uint32_t r1[4], r2[4], r3[4], q1[4], q2[4], q3[4]; };
__device__ __forceinline__ void ew8(const float (&x)[8], const float (&o)[8], const uint32_t* s, Ew8& w) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float o0 = o[2 * i], o1 = o[2 * i + 1];
        const float q0 = o0 > 0.f ? o0 * x[2 * i] : 0.f;
        const float q1 = o1 > 0.f ? o1 * x[2 * i + 1] : 0.f;
        const float r0 = o0 * __uint_as_float(s[2 * i]);          // S is finite: Omega == 0 gives exactly 0
        const float r1 = o1 * __uint_as_float(s[2 * i + 1]);
        split3_pair(q0, q1, w.q1[i], w.q2[i], w.q3[i]);
        split3_pair(r0, r1, w.r1[i], w.r2[i], w.r3[i]);
    }
}
// half h of a chunk's pieces -> TMEM: R1, R2 back over S in place (`zcol`), R3 and the Q pieces into the E block `ecol`
__device__ __forceinline__ void ew8_store(uint32_t zcol, uint32_t ecol, int h, const Ew8& w) {
    tmem_st4(zcol + 4 * h, w.r1); tmem_st4(zcol + 8 + 4 * h, w.r2);
    tmem_st4(ecol + O_R3 + 4 * h, w.r3); tmem_st4(ecol + O_Q1 + 4 * h, w.q1);
    tmem_st4(ecol + O_Q2 + 4 * h, w.q2); tmem_st4(ecol + O_Q3 + 4 * h, w.q3);
}

// ---------------------------------------------------------------- host: tensor maps
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time libcuda dependency)
typedef CUresult (*encode_fn_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline encode_fn_t encode_fn() {
    static encode_fn_t fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<encode_fn_t>(p);
    }
    return fn;
}

// 2-D fp32 map over a row-major [rows, P] array, box [box_rows][box_px], shared-memory swizzle 0 / 64 / 128 bytes
inline bool make_map(CUtensorMap* m, const float* base, long long rows, long long P, int box_rows, int box_px, int swizzle_bytes) {
    encode_fn_t fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)P, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)P * sizeof(float)};
    const cuuint32_t box[2] = {(cuuint32_t)box_px, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE,
              swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tc

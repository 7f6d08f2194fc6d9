// ann_bf16.cu -- K4: the ANN source term on the 5th-gen tensor cores (tcgen05.mma, fp32 accumulators in TMEM,
// weights streamed by TMA bulk copies): one persistent warp-specialised kernel for the whole chain
// (1600-800-400 GELU MLP; DESIGN.md section 6 "K4" and reading A21).
//
// Per 128-cell tile (UMMA M = 128, one cell per TMEM lane) a CTA runs
//   prologue   T, p, Y -> Box-Cox + z-score -> fp16 A0 [128 x 32] (+ two columns of ones for the biases) (threads)
//   phase A    for each half h of layer 2's outputs (N = d2/2 <= 400 TMEM columns):
//                D2 = A0 Wb2[h]^T                               (bias stage)                      (tcgen05)
//                for each 32-wide chunk c of layer 1:  D1 = A0 W1_c^T                              (tcgen05)
//                  an epilogue group: tcgen05.ld, GELU, fp16 -> A1 ring (128B-swizzled smem)       (threads)
//                  D2 += A1_c W2[h, c]^T                                                           (tcgen05)
//              drain D2: GELU, fp16 -> this CTA's private H2 scratch (global, L2-resident)
//   phase B    D3 = A0 Wb3^T + H2 W3^T with the H2 chunks read back by TMA; drain D3 in 64-wide chunks:
//              GELU, fp16 -> H3 ring -> D4 += H3_c W4_c^T; final epilogue: +b4, inverse Box-Cox, sum-to-one
//              renormalisation, rho, omega -> global (coalesced SoA).
// Layer 1 is recomputed for each half of layer 2 (K = 23: 2 % of the MMA work) because neither a 128 x 1600
// 16-bit activation tile (400 KB) nor a 128 x 800 fp32 accumulator (800 TMEM columns) fits on an SM.  All weights
// are re-tiled at create time into the exact 128B-swizzled K-major shared-memory images the UMMA descriptors
// expect, in streaming order, so every TMA transfer is one contiguous cp.async.bulk of 8-26 KB.
//
// Warp roles (20 warps): 0 = the two TMA producers (lane 0: weight ring; lane 1: W4, W1 quads, H2 chunks -- the two
// sides of one divergent branch), 1 and 3 = the two alternating layer-2/3 MMA issuers (warp 1 also issues layer 4),
// 2 = TMEM allocator and layer-1 MMA issuer, 4..15 = kGroups epilogue groups of four warps (warp w owns TMEM lanes
// 32 (w % 4) .. +31; group g takes every kGroups-th layer-1 chunk), 16..19 = four cell-I/O warps (next tile's
// Box-Cox features -> A0, previous tile's D4 -> inverse Box-Cox -> omega).
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <cstdlib>

#include <cstring>
#include <new>

#include "ann_common.cuh"

namespace {

// ---- geometry ---------------------------------------------------------------------------------
constexpr int kTileM = 128;
// Registers by role (setmaxnreg acts on a warpgroup = four consecutive warps; the launch gives every thread 96): warps 0..3
// (TMA producers, MMA issuers) keep 48, the three epilogue groups take 112 each -- 128 x (48 + 3 x 112 + 96) = 640 x 96.  The
// epilogue's GELU chains are what the kernel waits for; with 112 registers ptxas keeps more of them in flight (A/B on one box: 6.05 -> 5.88 ms,
// on another 6.14 -> 6.07; four groups of 88 or 96 registers: 5.95-5.99 ms on the first).
constexpr int kRegsIssue = 48, kRegsEpilogue = 112;
constexpr int kGroups = 3;                     // epilogue groups of 4 warps (one warp per TMEM lane quarter)
constexpr int kIssuer2Warp = 3;                // second layer-2/3 MMA issuer
constexpr int kIoWarp = 4 + 4 * kGroups;       // four cell-I/O warps: next tile's features -> A0, this tile's D4 -> omega
constexpr int kThreads = 32 * (kIoWarp + 4);
constexpr int kWStages = 4;
constexpr int kA1Tiles = 3;                 // [128 x 64] activation tiles of the A1 ring = 2 * kA1Tiles 32-column slots
constexpr int kA1Slots = 2 * kA1Tiles;
constexpr int kChunkBytes = kTileM * 128;  // one [128 x 64] bf16 K-major swizzled operand tile
constexpr int kW1QuadBytes = 64 * 128;     // four 32-row layer-1 chunks: [2 x 32 rows] x [2 x 32 K] bf16
constexpr int kSmallCol = 400;             // TMEM columns [400, 496): three 32-column D1 buffers (D4 reuses the first)
constexpr int kSmallBufs = 3;
constexpr int kTmemCols = 512;

struct NetGeom {
    int K, K0steps;          // species, k-steps (of 16) over the K+4 layer-1 inputs (features, 2 bias columns)
    int d1, d2, d3;          // hidden widths
    int NC;                  // d1 / 32 chunks of layer 1 (one 32-wide K stage of layer 2 each)
    int NH, na2, nb2;        // half of d2 and its two MMA N pieces
    int n3a, n3b;            // layer-3 N pieces
    int NKS;                 // d2 / 32 K-stages of layer 3
    int NKC;                 // ceil(d2 / 64) H2 chunks
    int NJ;                  // ceil(d3 / 64) H3 chunks
    int w2_tile_bytes, w3_tile_bytes, w_slot_bytes, w4_bytes;
    int smem_bytes;
    // shared-memory offsets (bytes from the 1024-aligned base)
    int off_w, off_r1, off_r2, off_w4, off_bar;
};

struct Bf16Dev {
    const uint8_t* w1t;  // [ceil(NC/4)][8192]
    const uint8_t* w2t;  // [2][NC][w2_tile_bytes]
    const uint8_t* w3t;  // [NKS][w3_tile_bytes]
    const uint8_t* w4t;  // [NJ][4096]
    const float *b1, *b2, *b3, *b4;
};

}  // namespace

struct Bf16Plan {
    NetGeom g;
    Bf16Dev d;
    float b4_host[32] = {0};
    void* blob = nullptr;
};

namespace {

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
        : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, 128B-swizzled operand tile: 8-row groups 1024 B apart (SBO), descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// kind::f16 instruction descriptor: D = f32 (bit 4), A and B = fp16 (format 0 in bits 7.. and 10..: kind::f16 wants
// both operands in one format, A21), both K-major, N >> 3 in bits 17.., M >> 4 in bits 24..
__device__ __forceinline__ uint32_t umma_idesc(int N) {
    return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .b32 rx;\n\t.reg .pred px;\n\t"
        "elect.sync rx|px, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, px;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    return done != 0;
}

// Non-suspending wait for the two producer lanes that share warp 0: a suspended try_wait of one lane would hold back
// the other lane's loop.
__device__ __forceinline__ void mbar_poll(uint32_t bar, uint32_t parity) {
    while (!mbar_test(bar, parity)) { }
}

__device__ __forceinline__ float tanh_approx(float x) {
    float r;
    asm("tanh.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// two fp32 -> packed fp16x2 (first argument in the low half = lower K index); saturates at +-65504 instead of inf
__device__ __forceinline__ uint32_t pack_act(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
// GELU (A13) of two fp32 accumulators -> packed fp16x2.  Tanh form v/2 (1 + tanh(sqrt(2/pi) (v + 0.044715 v^3))),
// evaluated in packed fp32 (FFMA2) with MUFU.TANH in fp32 (measured 3e-6 rms on this part) and rounded to fp16 once,
// at the end: next to an exactly rounded fp16 activation the only error left is that of the tanh form (<= 4.7e-4
// at |v| ~ 2-3, but third-order exact at v = 0 where the pre-activations live: it moves the network output by 3e-6
// rms against 2e-5 from the fp16 roundings).  A minimax refit of the two constants halves the maximum error and was
// tried: it is WORSE (its slope error at v = 0 is systematic and adds up coherently over 1600 units: 4.6e-5 rms at
// the output).  The earlier all-fp16x2 evaluation (fp16 v, three fp16 roundings inside the tanh argument,
// tanh.approx.f16x2) had 2-3x the rounding error of the result's own fp16 rounding, and its v*v overflowed for
// |v| > 255.
__device__ __forceinline__ uint32_t gelu_pair(float a, float b) {
    const float2 v = make_float2(a, b);
    const float2 t = __ffma2_rn(__fmul2_rn(v, v), make_float2(0.0356774081f, 0.0356774081f), make_float2(0.7978845608f, 0.7978845608f));
    const float2 u = __fmul2_rn(t, v);
    // the activation is held as 2 GELU(v) = v + v tanh(u): the factor 1/2 sits in the next layer's weights (exact: a power of
    // two), which saves one of eight instructions per pair
    const float2 r = __ffma2_rn(v, make_float2(tanh_approx(u.x), tanh_approx(u.y)), v);
    return pack_act(r.x, r.y);
}
// dY*_k of ann_common.cuh with MUFU-grade transcendentals (ex2/lg2/rcp.approx): 5 MUFU + a few FMA per species
// instead of powf/log1pf/expm1f (~400 instructions).  Its error (<= 2e-4 relative for |lambda Delta| >= 1e-3 Y^lambda)
// is far inside the 2e-2 budget of this path; the fp32 path (ann_fp32.cu) keeps the accurate form.
__device__ __forceinline__ float ann_dystar_fast(float y, float delta, float lambda, float inv_lambda) {
    // branch-free: y > 0: Y (2^(log2(1 + z)/lambda) - 1), z = lambda Delta / Y^lambda, Y* = 0 when z <= -1;
    //              y = 0: max(lambda Delta, 0)^(1/lambda)
    const float q = exp2f(lambda * __log2f(y));
    const float z = lambda * delta * rcp_approx(q);
    const float pos = y * (exp2f(__log2f(1.0f + z) * inv_lambda) - 1.0f);
    const float base = lambda * delta;
    const float zero = base > 0.f ? exp2f(__log2f(base) * inv_lambda) : 0.f;
    return y > 0.f ? ((z > -1.0f) ? pos : -y) : zero;
}
// byte offset of 16-byte chunk c16 (0..7) of row r inside a 128B-swizzled [rows x 64] bf16 tile
__device__ __forceinline__ uint32_t swz(int r, int c16) { return (uint32_t)(r * 128 + ((c16 ^ (r & 7)) << 4)); }

__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,"
        "%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}

// barrier indices
enum {
    B_W_FULL = 0, B_W_EMPTY = B_W_FULL + kWStages, B_W1_FULL = B_W_EMPTY + kWStages, B_W1_EMPTY = B_W1_FULL + 2,
    B_A0_FULL = B_W1_EMPTY + 2, B_SMALL_FULL, B_SMALL_EMPTY = B_SMALL_FULL + kGroups,
    B_A1_FULL = B_SMALL_EMPTY + kSmallBufs, B_A1_EMPTY = B_A1_FULL + kA1Slots, B_ACC_FULL = B_A1_EMPTY + kA1Slots, B_ACC_EMPTY,
    B_H2_FULL, B_H2C_FULL, B_H2C_EMPTY = B_H2C_FULL + 2, B_H3_FULL = B_H2C_EMPTY + 2, B_H3_EMPTY = B_H3_FULL + 2, B_TILE_DONE = B_H3_EMPTY + 2,
    B_W4_FULL, B_ACC_START, B_A0_EMPTY, B_COUNT
};

struct KArgs {
    NetGeom g;
    Bf16Dev d;
    float invW[32], b4[32];   // 1/W_k and the last layer's bias as constant-bank operands of the final epilogue
    long long n, ld;
    const float *T, *p, *Y;
    float *omega, *dY;
    float* raw;        // per-species-network mode (ann_mmlp.cu): the final epilogue only stores o[raw_row] + b4 to raw[raw_row][ld]
    int raw_row;
    uint8_t* scratch;  // gridDim.x * NKC * 16384 bytes
};

__global__ void __launch_bounds__(kThreads, 1)
ann_bf16_kernel(const __grid_constant__ KArgs a, const __grid_constant__ AnnNorm nm) {
    extern __shared__ uint8_t smem_dyn[];
    const NetGeom& g = a.g;
    const uint32_t sbase = (smem_u32(smem_dyn) + 1023u) & ~1023u;
    uint8_t* sgen = smem_dyn + (sbase - smem_u32(smem_dyn));
    const uint32_t s_w = sbase + g.off_w, s_r1 = sbase + g.off_r1, s_r2 = sbase + g.off_r2, s_w4 = sbase + g.off_w4;
    const uint32_t s_bar = sbase + g.off_bar;
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(sgen + g.off_bar + B_COUNT * 8);
    auto bar = [&](int i) { return s_bar + 8u * (uint32_t)i; };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long num_tiles = (a.n + kTileM - 1) / kTileM;

    if (threadIdx.x == 32) {
        for (int i = 0; i < B_COUNT; ++i) {
            uint32_t cnt = 1;
            if ((i >= B_SMALL_EMPTY && i < B_SMALL_EMPTY + kSmallBufs) || (i >= B_A1_FULL && i < B_A1_FULL + kA1Slots)) cnt = 4;
            if (i == B_ACC_EMPTY || i == B_H3_FULL || i == B_H3_FULL + 1) cnt = 4 * kGroups;
            if (i == B_A0_FULL) cnt = 4;
            if (i == B_H2_FULL) cnt = 8 * kGroups;
            if (i == B_ACC_FULL || i == B_H2C_EMPTY || i == B_H2C_EMPTY + 1) cnt = 2;  // one commit per issuer
            mbar_init(bar(i), cnt);
        }
        fence_barrier_init();
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         smem_u32((const void*)tmem_slot)),
                     "n"(kTmemCols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // register budget by role: kRegsIssue / kRegsEpilogue above (every warp of a warpgroup executes its setmaxnreg)

    if (warp == 0) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsIssue));
        // ================= TMA producers: two lanes of one warp, each with its own loop (the two sides of one divergent
        // branch make independent progress; 20 warps instead of 21 lifts the register cap from 80 to 96) =================
        // lane 0: weight ring
        if (lane == 0) {
            uint32_t cnt = 0;
            auto load = [&](const uint8_t* src, uint32_t bytes) {
                const uint32_t slot = cnt % kWStages, par = (cnt / kWStages) & 1;
                mbar_poll(bar(B_W_EMPTY + slot), par ^ 1);
                mbar_expect_tx(bar(B_W_FULL + slot), bytes);
                tma_bulk_g2s(s_w + slot * g.w_slot_bytes, src, bytes, bar(B_W_FULL + slot));
                ++cnt;
            };
            for (long long tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                const int n2 = 2 * (g.NC + 1);  // per half: the bias tile, then one tile per layer-1 chunk
                for (int i = 0; i < n2; ++i) load(a.d.w2t + (size_t)i * g.w2_tile_bytes, g.w2_tile_bytes);
                for (int ks = 0; ks <= g.NKS; ++ks) load(a.d.w3t + (size_t)ks * g.w3_tile_bytes, g.w3_tile_bytes);
            }
        } else if (lane == 1) {
            // lane 1: W4 (once), W1 quads, H2 chunks
            mbar_expect_tx(bar(B_W4_FULL), g.w4_bytes);
            tma_bulk_g2s(s_w4, a.d.w4t, g.w4_bytes, bar(B_W4_FULL));
            const uint8_t* scratch = a.scratch + (size_t)blockIdx.x * g.NKC * kChunkBytes;
            const int nquads = (g.NC + 3) / 4;
            uint32_t w1c = 0, h2c = 0, tc = 0;
            for (long long tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tc) {
                for (int h = 0; h < 2; ++h)
                    for (int qd = 0; qd < nquads; ++qd, ++w1c) {
                        const uint32_t slot = w1c & 1, par = (w1c >> 1) & 1;
                        mbar_poll(bar(B_W1_EMPTY + slot), par ^ 1);
                        mbar_expect_tx(bar(B_W1_FULL + slot), kW1QuadBytes);
                        tma_bulk_g2s(s_r2 + kChunkBytes + slot * kW1QuadBytes, a.d.w1t + (size_t)qd * kW1QuadBytes,
                                     kW1QuadBytes, bar(B_W1_FULL + slot));
                    }
                mbar_poll(bar(B_H2_FULL), tc & 1);  // both halves of H2 are in the scratch
                for (int kc = 0; kc < g.NKC; ++kc, ++h2c) {
                    const uint32_t slot = h2c & 1, par = (h2c >> 1) & 1;
                    mbar_poll(bar(B_H2C_EMPTY + slot), par ^ 1);
                    mbar_expect_tx(bar(B_H2C_FULL + slot), kChunkBytes);
                    tma_bulk_g2s(s_r1 + slot * kChunkBytes, scratch + (size_t)kc * kChunkBytes, kChunkBytes,
                                 bar(B_H2C_FULL + slot));
                }
            }
        }
    } else if (warp == 2) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsIssue));
        // ================= layer-1 MMA issuer (this warp also owns the TMEM allocation) =================
        // Layer 1 has its own issuing warp so that neither issuer has more than two mbarrier round trips per
        // 32-column chunk: it runs ahead of layer 2 as far as the three D1 buffers allow.  Whole warp convergent,
        // one elected lane issues (ptxas then keeps descriptors and barrier addresses in uniform registers).
        const uint32_t id32 = umma_idesc(32);
        const uint64_t dA0 = umma_desc(s_r2), dW1 = umma_desc(s_r2 + kChunkBytes);
        uint32_t w1c = 0, gs = 0, ac = 0, tc = 0;
        for (long long tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tc) {
            mbar_wait(bar(B_A0_FULL), tc & 1);
            for (int h = 0; h < 2; ++h)
                for (int c = 0; c < g.NC; ++c, ++gs, ++ac) {
                    const uint32_t slot = w1c & 1, sb = gs % kSmallBufs;
                    if ((c & 3) == 0) mbar_wait(bar(B_W1_FULL + slot), (w1c >> 1) & 1);
                    mbar_wait(bar(B_SMALL_EMPTY + sb), ((gs / kSmallBufs) & 1) ^ 1);
                    tc_fence_after();
                    const bool quad_done = (c & 3) == 3 || c == g.NC - 1;
                    if (elect_one()) {
                        const uint64_t b0 = dW1 + ((slot * kW1QuadBytes + ((c & 3) >> 1) * 4096 + (c & 1) * 64) >> 4);
                        const uint32_t dd = tmem + kSmallCol + sb * 32;
                        tc_mma(dd, dA0, b0, id32, 0u);
                        if (g.K0steps > 1) tc_mma(dd, dA0 + 2, b0 + 2, id32, 1u);
                        tc_commit(bar(B_SMALL_FULL + ac % kGroups));
                        if (quad_done) tc_commit(bar(B_W1_EMPTY + slot));
                    }
                    __syncwarp();
                    if (quad_done) ++w1c;
                }
            ++gs;  // the D4 accumulation of this tile (issued by warp 1) takes the next buffer of the ring
        }
    } else if (warp == 1 || warp == kIssuer2Warp) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsIssue));
        // ================= layer-2/3/4 MMA issuers (two warps, each convergent, one elected lane issues) ============
        // One warp needs ~700 cycles of its own instruction stream per 32-wide K stage (two mbarrier round trips,
        // four UTCHMMA, two UTCBAR, warp re-convergence) against ~460 cycles of tensor time, so the stages of the
        // weight ring alternate between two issuing warps: stage st goes to issuer st & 1.  The first stage of every
        // accumulation (the bias stage, accumulate = 0) is announced on B_ACC_START before the other issuer adds to it;
        // barriers that follow a whole accumulation / H2 tile (ACC_FULL, H2C_EMPTY) take one commit from each issuer.
        const int id = (warp == 1) ? 0 : 1;
        const uint32_t id32 = umma_idesc(32);
        const uint32_t id2a = umma_idesc(g.na2), id2b = umma_idesc(g.nb2 > 0 ? g.nb2 : 16);
        const uint32_t id3a = umma_idesc(g.n3a), id3b = umma_idesc(g.n3b > 0 ? g.n3b : 16);
        const uint64_t dR2 = umma_desc(s_r2), dR1 = umma_desc(s_r1), dW = umma_desc(s_w), dW4 = umma_desc(s_w4);
        const uint32_t w_slot16 = (uint32_t)g.w_slot_bytes >> 4;
        // st: stages of the weight ring; gs: uses of the small-accumulator ring; ac: uses of the A1 slots;
        // acc: accumulations started (three per tile)
        uint32_t st = 0, gs = 0, ac = 0, ae = 0, h2cc = 0, h3c = 0, tc = 0, acc = 0;

        auto issue_stage = [&](uint64_t ad, int na, int nb, uint32_t ida, uint32_t idb, bool first, uint32_t extra) {
            const uint32_t slot = st % kWStages;
            mbar_wait(bar(B_W_FULL + slot), (st / kWStages) & 1);
            tc_fence_after();
            if (elect_one()) {
                const uint64_t wb = dW + slot * w_slot16;
                tc_mma(tmem, ad, wb, ida, first ? 0u : 1u);
                if (nb > 0) tc_mma(tmem + na, ad, wb + 4, idb, first ? 0u : 1u);
                tc_mma(tmem, ad + 2, wb + 2, ida, 1u);
                if (nb > 0) tc_mma(tmem + na, ad + 2, wb + 6, idb, 1u);
                tc_commit(bar(B_W_EMPTY + slot));
                if (extra) tc_commit(extra);
            }
            __syncwarp();
        };
        // bias stage of an accumulation: whoever owns stage st issues it and announces it; the other waits
        auto start_acc = [&](int na, int nb, uint32_t ida, uint32_t idb, uint32_t extra) {
            if ((int)(st & 1) == id) {
                mbar_wait(bar(B_ACC_EMPTY), (ae & 1) ^ 1);
                issue_stage(dR2, na, nb, ida, idb, true, extra);
                if (lane == 0) mbar_arrive(bar(B_ACC_START));
            } else {
                mbar_wait(bar(B_ACC_START), acc & 1);
            }
            ++ae;
            ++acc;
            ++st;
        };

        for (long long tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tc) {
            mbar_wait(bar(B_A0_FULL), tc & 1);
            // ---- phase A: layer 2, one half of its outputs at a time, one stage per layer-1 chunk ----
            for (int h = 0; h < 2; ++h) {
                start_acc(g.na2, g.nb2, id2a, id2b, 0u);
                for (int c = 0; c < g.NC; ++c, ++ac, ++st) {
                    if ((int)(st & 1) != id) continue;
                    const uint32_t slot = ac % kA1Slots;
                    mbar_wait(bar(B_A1_FULL + slot), (ac / kA1Slots) & 1);
                    issue_stage(dR1 + (((slot >> 1) * kChunkBytes + (slot & 1) * 64) >> 4), g.na2, g.nb2, id2a, id2b, false,
                                bar(B_A1_EMPTY + slot));
                }
                if (elect_one()) tc_commit(bar(B_ACC_FULL));
                __syncwarp();
            }
            gs += 2 * g.NC;
            // ---- phase B: layer 3 from the H2 chunks, then layer 4 fed by the D3 drain ----
            start_acc(g.n3a, g.n3b, id3a, id3b, bar(B_A0_EMPTY));   // last use of A0: the I/O warps may write the next tile's
            for (int ks = 0; ks < g.NKS; ++ks, ++st) {
                const uint32_t slot = h2cc & 1;
                const bool last = (ks & 1) == 1 || ks == g.NKS - 1;
                if ((int)(st & 1) == id) {
                    mbar_wait(bar(B_H2C_FULL + slot), (h2cc >> 1) & 1);
                    issue_stage(dR1 + ((slot * kChunkBytes + (ks & 1) * 64) >> 4), g.n3a, g.n3b, id3a, id3b, false, 0u);
                }
                if (last) {   // both issuers commit once per H2 tile (a commit with nothing outstanding arrives at once)
                    if (elect_one()) tc_commit(bar(B_H2C_EMPTY + slot));
                    __syncwarp();
                    ++h2cc;
                }
            }
            if (elect_one()) tc_commit(bar(B_ACC_FULL));
            __syncwarp();
            const uint32_t sb = gs % kSmallBufs;
            if (id == 0) {
                if (tc == 0) mbar_wait(bar(B_W4_FULL), 0);
                for (int jj = 0; jj < g.NJ; ++jj, ++h3c) {
                    const uint32_t slot = h3c & 1;
                    mbar_wait(bar(B_H3_FULL + slot), (h3c >> 1) & 1);
                    if (jj == 0) mbar_wait(bar(B_SMALL_EMPTY + sb), ((gs / kSmallBufs) & 1) ^ 1);
                    tc_fence_after();
                    if (elect_one()) {
                        const int ksteps = min(64, g.d3 - jj * 64) / 16;
                        const uint64_t ha = dR1 + ((slot * kChunkBytes) >> 4), wa = dW4 + ((jj * 4096) >> 4);
                        for (int kk = 0; kk < ksteps; ++kk)
                            tc_mma(tmem + kSmallCol + sb * 32, ha + 2 * kk, wa + 2 * kk, id32, (jj > 0 || kk > 0) ? 1u : 0u);
                        tc_commit(bar(B_H3_EMPTY + slot));
                    }
                    __syncwarp();
                }
                if (elect_one()) {
                    tc_commit(bar(B_TILE_DONE));   // D4 is complete: the final epilogue may read it, R2 is free
                }
                __syncwarp();
            }
            ++gs;
        }
    } else if (warp >= 4 && warp < 4 + 4 * kGroups) {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsEpilogue));
        // ================= epilogue warps: kGroups groups of four (one warp per TMEM lane quarter) =================
        // Group grp takes every kGroups-th layer-1 chunk (so several chunks are in flight), every kGroups-th
        // 16-column unit of the D2/D3 drains, and one 16-byte column chunk of the A0 feature tile.
        const int ew = warp - 4, q = ew & 3, grp = ew >> 2;
        const int row = q * 32 + lane;
        const uint32_t t_lane = tmem + ((uint32_t)(q * 32) << 16);
        uint8_t* scratch = a.scratch + (size_t)blockIdx.x * g.NKC * kChunkBytes;
        uint32_t gs = 0, ac = 0, af = 0, h3c = 0;

        auto st_shared16 = [&](uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
        };
        // GELU on 16 accumulators (biases are already in them) -> 8 packed fp16x2 words
        auto gelu16 = [&](const uint32_t* r, uint32_t (&o)[8]) {
#pragma unroll
            for (int i = 0; i < 8; ++i) o[i] = gelu_pair(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1]));
        };

        uint32_t tcnt = 0;
        for (long long tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcnt) {
            // the H3 ring lives in R1: the previous tile's layer-4 MMAs must be done before A1 chunks go there again
            if (tcnt > 0) mbar_wait(bar(B_TILE_DONE), (tcnt - 1) & 1);
            // ---- phase A ----
            for (int h = 0; h < 2; ++h) {
                for (int c = 0; c < g.NC; ++c, ++gs, ++ac) {
                    if ((int)(ac % kGroups) != grp) continue;
                    const uint32_t sb = gs % kSmallBufs;
                    mbar_wait(bar(B_SMALL_FULL + grp), (ac / kGroups) & 1);
                    tc_fence_after();
                    uint32_t r[32];
                    tc_ld32(t_lane + kSmallCol + sb * 32, r);
                    tc_wait_ld();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_SMALL_EMPTY + sb));
                    uint32_t o[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i)   // b1 is already in the accumulator (bias columns of W1)
                        o[i] = gelu_pair(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1]));
                    const uint32_t slot = ac % kA1Slots;
                    mbar_wait(bar(B_A1_EMPTY + slot), ((ac / kA1Slots) & 1) ^ 1);
                    const uint32_t base = s_r1 + (slot >> 1) * kChunkBytes;
#pragma unroll
                    for (int c4 = 0; c4 < 4; ++c4)
                        st_shared16(base + swz(row, (slot & 1) * 4 + c4), o[4 * c4], o[4 * c4 + 1], o[4 * c4 + 2], o[4 * c4 + 3]);
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar(B_A1_FULL + slot));
                }
                // drain D2 (this half): +b2, GELU, fp16 -> H2 scratch in the chunk images phase B loads
                mbar_wait(bar(B_ACC_FULL), af & 1);
                ++af;
                tc_fence_after();
                {
                    // software-pipelined: the TMEM load of the next 16-column unit is in flight during the math
                    auto store_unit = [&](const uint32_t* r, int c0) {
                        uint32_t o[8];
                        gelu16(r, o);
                        const int gc = h * g.NH + c0;
                        uint8_t* dst = scratch + (size_t)(gc >> 6) * kChunkBytes;
                        const int c16 = (gc & 63) >> 3;
                        // the two 16-byte chunks of a 16-column unit share one 32-byte sector of the swizzled row (their
                        // order inside it depends on the row parity): one 256-bit store instead of two scattered 128-bit ones
                        const bool sw = row & 1;
                        uint8_t* d32 = dst + row * 128 + (((c16 ^ (row & 7)) & ~1) << 4);
                        asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(d32), "r"(sw ? o[4] : o[0]),
                                     "r"(sw ? o[5] : o[1]), "r"(sw ? o[6] : o[2]), "r"(sw ? o[7] : o[3]), "r"(sw ? o[0] : o[4]),
                                     "r"(sw ? o[1] : o[5]), "r"(sw ? o[2] : o[6]), "r"(sw ? o[3] : o[7])
                                     : "memory");
                    };
                    constexpr int kStep = 16 * kGroups;
                    uint32_t ra[16], rb[16];
                    int c0 = grp * 16;
                    if (c0 < g.NH) tc_ld16(t_lane + c0, ra);
                    while (c0 < g.NH) {
                        tc_wait_ld();
                        if (c0 + kStep < g.NH) tc_ld16(t_lane + c0 + kStep, rb);
                        store_unit(ra, c0);
                        c0 += kStep;
                        if (c0 >= g.NH) break;
                        tc_wait_ld();
                        if (c0 + kStep < g.NH) tc_ld16(t_lane + c0 + kStep, ra);
                        store_unit(rb, c0);
                        c0 += kStep;
                    }
                }
                tc_fence_before();
                // generic-proxy stores to the scratch -> async-proxy (TMA) reads by warp 3 of this CTA: the proxy fence for
                // the global space, then the release/acquire pair of the mbarrier.  (A preceding __threadfence and the
                // all-spaces form of the fence add a MEMBAR.SC.GPU + ERRBAR: 2 % of the kernel.)
                fence_proxy_async_global();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(bar(B_ACC_EMPTY));
                    mbar_arrive(bar(B_H2_FULL));
                }
            }
            // ---- phase B: drain D3 in 64-wide chunks -> H3 ring (feeds layer 4); group grp owns 16-column unit grp ----
            mbar_wait(bar(B_ACC_FULL), af & 1);
            ++af;
            tc_fence_after();
            for (int jj = 0; jj < g.NJ; ++jj, ++h3c) {
                // the four 16-column units of this 64-wide chunk go round-robin over the groups, continuing from the
                // previous chunk (unit jj * 4 + u -> group (jj * 4 + u) % kGroups): one or two per group, balanced
                const int u0 = (grp + kGroups * 4 - (jj * 4) % kGroups) % kGroups;
                uint32_t o[2][8];
                bool have[2];
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int u = u0 + i * kGroups, c0 = jj * 64 + u * 16;
                    have[i] = u < 4 && c0 < g.d3;
                    if (have[i]) {
                        uint32_t r[16];
                        tc_ld16(t_lane + c0, r);
                        tc_wait_ld();
                        gelu16(r, o[i]);
                    }
                }
                const uint32_t slot = h3c & 1;
                mbar_wait(bar(B_H3_EMPTY + slot), ((h3c >> 1) & 1) ^ 1);
                const uint32_t base = s_r1 + slot * kChunkBytes;   // R1 is idle once layer 3 has completed
#pragma unroll
                for (int i = 0; i < 2; ++i)
                    if (have[i]) {
                        const int u = u0 + i * kGroups;
                        st_shared16(base + swz(row, u * 2), o[i][0], o[i][1], o[i][2], o[i][3]);
                        st_shared16(base + swz(row, u * 2 + 1), o[i][4], o[i][5], o[i][6], o[i][7]);
                    }
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_H3_FULL + slot));
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_ACC_EMPTY));
            ++gs;   // the D4 accumulation of this tile takes the next buffer of the small ring (read by the I/O warps)
        }
    } else if (warp >= kIoWarp && warp < kIoWarp + 4) {
        // ================= cell-I/O warps: one thread per row of the tile =================
        // They run one tile ahead on the input side (T, p, Y -> Box-Cox features -> A0) and one tile behind on the
        // output side (D4 -> Delta -> inverse Box-Cox -> renormalise -> omega, A9-A11, A17), so that neither the
        // global-memory latency of the cell data nor the MUFU chains of the final epilogue sit between two tiles' MMAs.
        const int q = warp & 3, row = q * 32 + lane;
        const uint32_t t_lane = tmem + ((uint32_t)(q * 32) << 16);
        const float lam = nm.lambda, inv_lam = nm.inv_lambda;

        // features of one cell + two bias columns of ones -> 16 packed fp16x2 words (one A0 row)
        auto features = [&](long long tile, uint32_t (&o)[16]) {
            const long long cell = tile * kTileM + row;
            const bool valid = cell < a.n;
            const long long cl = valid ? cell : 0;
            float raw[32];
#pragma unroll
            for (int f = 0; f < 32; ++f)
                raw[f] = (f == 0) ? __ldg(a.T + cl) : (f == 1) ? __ldg(a.p + cl)
                       : (f < g.K + 2) ? __ldg(a.Y + (size_t)(f - 2) * a.ld + cl) : 0.f;
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                float v[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int f = 2 * i + e;
                    float x = 0.f;
                    if (f < g.K + 2) {
                        if (valid) {
                            if (f < 2) x = (raw[f] - nm.x_mean[f]) * nm.x_inv_std[f];
                            else {
                                const float qy = exp2f(lam * __log2f(raw[f]));  // y^lambda, 0 -> 0
                                x = ((qy - 1.0f) * inv_lam - nm.x_mean[f]) * nm.x_inv_std[f];
                            }
                        }
                    } else if (f < g.K + 4) {
                        x = 1.0f;  // multiplies the hi / lo parts of b1 (and b2, b3) stored as weight columns K+2, K+3
                    }
                    v[e] = x;
                }
                o[i] = pack_act(v[0], v[1]);
            }
        };
        auto write_a0 = [&](const uint32_t (&o)[16]) {
#pragma unroll
            for (int fc = 0; fc < 4; ++fc)
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(s_r2 + swz(row, fc)), "r"(o[4 * fc]),
                             "r"(o[4 * fc + 1]), "r"(o[4 * fc + 2]), "r"(o[4 * fc + 3])
                             : "memory");
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_A0_FULL));
        };

        uint32_t tcnt = 0, gs = 0;
        {
            uint32_t o[16];
            if ((long long)blockIdx.x < num_tiles) {
                features(blockIdx.x, o);
                write_a0(o);
            }
        }
        for (long long tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++tcnt) {
            const long long next = tile + gridDim.x;
            if (next < num_tiles) {
                uint32_t o[16];
                features(next, o);
                mbar_wait(bar(B_A0_EMPTY), tcnt & 1);   // layer 3's bias stage was the last reader of this tile's A0
                write_a0(o);
            }
            gs += 2 * g.NC;
            const uint32_t sb = gs % kSmallBufs;
            ++gs;
            const long long cell = tile * kTileM + row;
            const bool valid = cell < a.n;
            const long long cl = valid ? cell : 0;
            const float T = __ldg(a.T + cl), p = __ldg(a.p + cl);
            mbar_wait(bar(B_TILE_DONE), tcnt & 1);
            tc_fence_after();
            uint32_t r[32];
            tc_ld32(t_lane + kSmallCol + sb * 32, r);
            tc_wait_ld();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SMALL_EMPTY + sb));
            if (a.raw) {   // kernel-uniform: this launch is one of K one-output networks; the shared epilogue runs afterwards
                float o = 0.f;
#pragma unroll
                for (int k = 0; k < 32; ++k)
                    if (k == a.raw_row) o = __uint_as_float(r[k]) + a.b4[k];
                if (valid) a.raw[(size_t)a.raw_row * a.ld + cell] = o;
                continue;
            }
            // first pass: dY*_k (kept in r[k]), sum Y, sum dY*, 1 / Wbar; branch-free so the MUFU chains interleave
            float sumY = 0.f, sumd = 0.f, inv_Wbar = 0.f;
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                const bool on = k < g.K;
                const int kc = on ? k : 0;
                const float y = on ? __ldg(a.Y + (size_t)kc * a.ld + cl) : 0.f;
                sumY += y;
                inv_Wbar = fmaf(y, a.invW[kc], inv_Wbar);
                const float d = ann_dystar_fast(y, fmaf(nm.u_std[kc], __uint_as_float(r[k]) + a.b4[kc], nm.u_mean[kc]), lam, inv_lam);
                r[k] = __float_as_uint(on ? d : 0.f);
                sumd += __uint_as_float(r[k]);
            }
            // S - 1 = (sum Y - 1) + sum dY*: both terms are small and well conditioned in fp32 on this 2e-2 path
            const float Sm1 = (sumY - 1.0f) + sumd, inv_S = 1.0f / (1.0f + Sm1);
            const float rho_dt = p / (inv_Wbar * (float)DF_R_UNIVERSAL * T) * nm.inv_dt;
            if (valid) {
#pragma unroll
                for (int k = 0; k < 32; ++k) {
                    if (k < g.K) {
                        const float y = __ldg(a.Y + (size_t)k * a.ld + cell);   // L2 hit; off the critical path here
                        const float d = (__uint_as_float(r[k]) - y * Sm1) * inv_S;
                        if (a.dY) a.dY[(size_t)k * a.ld + cell] = d;
                        if (a.omega) a.omega[(size_t)k * a.ld + cell] = rho_dt * d;
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols));
    }
}

}  // namespace

// ---- host side: geometry, weight re-tiling, launch ------------------------------------------------
namespace {

uint16_t fp16_bits(float x) {  // round to nearest even, via the compiler's __half conversion on the host
    const __half h = __float2half_rn(x);
    uint16_t b;
    memcpy(&b, &h, 2);
    return b;
}
float fp16_value(float x) {
    const __half h = __float2half_rn(x);
    return __half2float(h);
}

// element (row r, column c < 64) of a 128B-swizzled K-major fp16 tile
inline void put(uint8_t* tile, int r, int c, float v) {
    const size_t off = (size_t)r * 128 + (size_t)((((c >> 3) ^ (r & 7)) << 4) + (c & 7) * 2);
    const uint16_t b = fp16_bits(v);
    memcpy(tile + off, &b, 2);
}

void split_n(int N, int* na, int* nb) {
    *na = ((N / 2 + 15) / 16) * 16;
    if (*na > N) *na = N;
    *nb = N - *na;
}

}  // namespace

df_status ann_bf16_create(df_ann* ann, const float* const* W, const float* const* b) {
    if (ann->n_layers != 4) return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: n_layers must be 4 (got %d)", ann->n_layers);
    const int K = ann->K, d1 = ann->dims[1], d2 = ann->dims[2], d3 = ann->dims[3];
    if (K > 28) return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: K <= 28 (got %d)", K);
    if (d1 % 64 || d1 < 64) return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: dims[1] %% 64 == 0 (got %d)", d1);
    if (d2 % 32 || d2 < 64 || d2 > 800) return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: dims[2] %% 32 == 0, 64..800 (got %d)", d2);
    if (d3 % 16 || d3 < 32 || d3 > 400) return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: dims[3] %% 16 == 0, 32..400 (got %d)", d3);

    // The contract of precision 1 (include/df_thermo.h): weights are bf16-valued and, like the biases, inside the
    // fp16 range, because the tensor path holds them in fp16 (A21; layers 2-4 halved, see gelu_pair) -- exact for bf16
    // values in [2^-14, 65504], within 2^-25 absolute below that.  Anything else would be re-rounded silently (or become inf): refuse it.
    for (int l = 0; l < 4; ++l) {
        const size_t nw = (size_t)ann->dims[l] * ann->dims[l + 1];
        for (size_t i = 0; i < nw; ++i) {
            const float w = W[l][i];
            uint32_t bits;
            memcpy(&bits, &w, 4);
            if (!(fabsf(w) <= 65504.0f))
                return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: W[%d][%zu] = %g is outside the fp16 range the tensor path holds weights in", l, i, (double)w);
            if (bits & 0xFFFFu)
                return df_set_error(DF_ERR_INVALID_ARG, "bf16 path: W[%d][%zu] = %.9g is not bf16-valued (round the weights to bf16 first)", l, i, (double)w);
        }
        for (int i = 0; i < ann->dims[l + 1]; ++i)
            if (!(fabsf(b[l][i]) <= 65504.0f))
                return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: b[%d][%d] = %g is outside the fp16 range", l, i, (double)b[l][i]);
    }

    Bf16Plan* P = new (std::nothrow) Bf16Plan;
    if (!P) return df_set_error(DF_ERR_ALLOC, "bf16 path: out of host memory");
    ann->bf16 = P;
    NetGeom& g = P->g;
    g.K = K;
    g.K0steps = (K + 4 <= 16) ? 1 : 2;  // features + 2 bias columns, fp16
    g.d1 = d1; g.d2 = d2; g.d3 = d3;
    g.NC = d1 / 32;
    g.NH = d2 / 2;
    split_n(g.NH, &g.na2, &g.nb2);
    split_n(d3, &g.n3a, &g.n3b);
    g.NKS = d2 / 32;
    g.NKC = (d2 + 63) / 64;
    g.NJ = (d3 + 63) / 64;
    g.w2_tile_bytes = g.na2 * 128;
    g.w3_tile_bytes = g.n3a * 128;
    g.w_slot_bytes = (g.w2_tile_bytes > g.w3_tile_bytes ? g.w2_tile_bytes : g.w3_tile_bytes);
    g.w_slot_bytes = (g.w_slot_bytes + 1023) / 1024 * 1024;
    g.w4_bytes = g.NJ * 4096;
    g.off_w = 0;
    g.off_r1 = kWStages * g.w_slot_bytes;
    g.off_r2 = g.off_r1 + kA1Tiles * kChunkBytes;
    g.off_w4 = g.off_r2 + 2 * kChunkBytes;
    g.off_bar = g.off_w4 + g.w4_bytes;
    g.smem_bytes = g.off_bar + B_COUNT * 8 + 16 + 1024;
    if (g.smem_bytes > 227 * 1024) return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path: layer widths need %d B of shared memory", g.smem_bytes);

    const int nquads = (g.NC + 3) / 4;
    const size_t sz_w1 = (size_t)nquads * kW1QuadBytes, sz_w2 = (size_t)2 * (g.NC + 1) * g.w2_tile_bytes,
                 sz_w3 = (size_t)(g.NKS + 1) * g.w3_tile_bytes, sz_w4 = (size_t)g.w4_bytes;
    const size_t sz_b = (size_t)(d1 + d2 + d3 + 32) * sizeof(float);
    const size_t o_w1 = 0, o_w2 = o_w1 + sz_w1, o_w3 = o_w2 + sz_w2, o_w4 = o_w3 + sz_w3, o_b = o_w4 + sz_w4;
    std::vector<uint8_t> blob(o_b + sz_b, 0);
    const int din = K + 2;
    // a bias rides in the accumulator as two weight columns (fp16 hi + lo parts) against the ones columns of A0
    auto put_bias = [&](uint8_t* t, int r, int col0, float bv) {
        const float hf = fp16_value(bv);
        put(t, r, col0 + din, hf);
        put(t, r, col0 + din + 1, bv - hf);
    };
    // W1: chunk c (32 outputs) sits in quad c/4 at rows 32*((c&3)>>1).., K columns 32*(c&1)..; columns K+2 and
    // K+3 carry the fp16 hi and lo parts of b1 (the A0 tile holds 1.0 there).
    for (int c = 0; c < g.NC; ++c) {
        uint8_t* t = blob.data() + o_w1 + (size_t)(c >> 2) * kW1QuadBytes;
        const int r0 = ((c & 3) >> 1) * 32, k0 = (c & 1) * 32;
        for (int r = 0; r < 32; ++r) {
            const int o = c * 32 + r;
            for (int k = 0; k < din; ++k) put(t, r0 + r, k0 + k, W[0][(size_t)o * din + k]);
            put_bias(t, r0 + r, k0, b[0][o]);
        }
    }
    // bias tiles: zero except K rows din, din + 1 (the ones columns of A0) = hi / lo parts of the bias
    for (int h = 0; h < 2; ++h) {
        uint8_t* t = blob.data() + o_w2 + (size_t)(h * (g.NC + 1)) * g.w2_tile_bytes;
        for (int r = 0; r < g.na2; ++r) put_bias(t, r, 0, b[1][h * g.NH + r]);
        for (int r = 0; r < g.nb2; ++r) put_bias(t, r, 32, b[1][h * g.NH + g.na2 + r]);
    }
    {
        uint8_t* t = blob.data() + o_w3;
        for (int r = 0; r < g.n3a; ++r) put_bias(t, r, 0, b[2][r]);
        for (int r = 0; r < g.n3b; ++r) put_bias(t, r, 32, b[2][g.n3a + r]);
    }
    // layers 2-4 read activations held as 2 GELU (gelu_pair): their weights are stored halved (the bias tiles are not: they
    // multiply the ones columns of A0)
    for (int h = 0; h < 2; ++h)
        for (int c = 0; c < g.NC; ++c) {
            uint8_t* t = blob.data() + o_w2 + (size_t)(h * (g.NC + 1) + 1 + c) * g.w2_tile_bytes;
            const int k0 = c * 32;
            for (int kk = 0; kk < 32; ++kk) {
                for (int r = 0; r < g.na2; ++r) put(t, r, kk, 0.5f * W[1][(size_t)(h * g.NH + r) * d1 + k0 + kk]);
                for (int r = 0; r < g.nb2; ++r) put(t, r, 32 + kk, 0.5f * W[1][(size_t)(h * g.NH + g.na2 + r) * d1 + k0 + kk]);
            }
        }
    for (int ks = 0; ks < g.NKS; ++ks) {
        uint8_t* t = blob.data() + o_w3 + (size_t)(ks + 1) * g.w3_tile_bytes;
        for (int kk = 0; kk < 32; ++kk) {
            for (int r = 0; r < g.n3a; ++r) put(t, r, kk, 0.5f * W[2][(size_t)r * d2 + ks * 32 + kk]);
            for (int r = 0; r < g.n3b; ++r) put(t, r, 32 + kk, 0.5f * W[2][(size_t)(g.n3a + r) * d2 + ks * 32 + kk]);
        }
    }
    for (int jj = 0; jj < g.NJ; ++jj) {
        uint8_t* t = blob.data() + o_w4 + (size_t)jj * 4096;
        for (int r = 0; r < K; ++r)
            for (int c = 0; c < 64 && jj * 64 + c < d3; ++c) put(t, r, c, 0.5f * W[3][(size_t)r * d3 + jj * 64 + c]);
    }
    float* hb = reinterpret_cast<float*>(blob.data() + o_b);
    memcpy(hb, b[0], sizeof(float) * d1);
    memcpy(hb + d1, b[1], sizeof(float) * d2);
    memcpy(hb + d1 + d2, b[2], sizeof(float) * d3);
    memcpy(hb + d1 + d2 + d3, b[3], sizeof(float) * K);
    memcpy(P->b4_host, b[3], sizeof(float) * K);

    if (cudaMalloc(&P->blob, blob.size()) != cudaSuccess) return df_set_error(DF_ERR_ALLOC, "bf16 path: cudaMalloc of %zu bytes failed", blob.size());
    DF_CUDA_TRY(cudaMemcpy(P->blob, blob.data(), blob.size(), cudaMemcpyHostToDevice));
    const uint8_t* base = static_cast<const uint8_t*>(P->blob);
    P->d.w1t = base + o_w1;
    P->d.w2t = base + o_w2;
    P->d.w3t = base + o_w3;
    P->d.w4t = base + o_w4;
    const float* db = reinterpret_cast<const float*>(base + o_b);
    P->d.b1 = db;
    P->d.b2 = db + d1;
    P->d.b3 = db + d1 + d2;
    P->d.b4 = db + d1 + d2 + d3;
    return DF_OK;
}

void ann_bf16_destroy(df_ann* ann) {
    if (!ann->bf16) return;
    cudaFree(ann->bf16->blob);
    delete ann->bf16;
    ann->bf16 = nullptr;
}

// one CTA per SM of the device the call runs on (persistent kernel), fewer when there are fewer tiles
static long long bf16_grid(long long n) {
    const long long tiles = (n + kTileM - 1) / kTileM;
    const int sms = df_device_sm_count();
    return tiles < sms ? tiles : (sms > 0 ? sms : 1);
}

size_t ann_bf16_workspace(const df_ann* ann, long long n) {
    return (size_t)bf16_grid(n) * ann->bf16->g.NKC * kChunkBytes;
}

df_status launch_ann_bf16(const df_ann* ann, const df_mech* mech, long long n, long long ld, const float* T,
                          const float* p, const float* Y, float* omega, float* dY, void* ws, size_t ws_bytes,
                          cudaStream_t s, float* raw, int raw_row) {
    const Bf16Plan* P = ann->bf16;
    const long long grid = bf16_grid(n);
    if (ws_bytes < (size_t)grid * P->g.NKC * kChunkBytes)
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source: workspace too small for this device");
    static DfPerDevice smem_attr;   // the attribute is per device; every handle shape fits the fixed maximum
    df_status st = df_ensure_dyn_smem((const void*)ann_bf16_kernel, 227 * 1024, &smem_attr);
    if (st != DF_OK) return st;
    KArgs a;
    a.g = P->g;
    a.d = P->d;
    for (int k = 0; k < 32; ++k) a.invW[k] = k < mech->K ? (float)(1.0 / mech->W_host[k]) : 0.f;
    memcpy(a.b4, P->b4_host, sizeof(a.b4));
    a.n = n;
    a.ld = ld;
    a.T = T; a.p = p; a.Y = Y;
    a.omega = omega; a.dY = dY;
    a.raw = raw; a.raw_row = raw_row;
    a.scratch = static_cast<uint8_t*>(ws);
    ann_bf16_kernel<<<(unsigned)grid, kThreads, P->g.smem_bytes, s>>>(a, ann->norm);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

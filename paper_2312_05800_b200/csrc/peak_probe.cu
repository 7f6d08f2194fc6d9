// peak_probe.cu -- measurement helper, not part of the hot path: the FP32 FMA-pipe peak the property kernels' "alu"
// roofline is quoted against ("the bench must measure an FFMA-chain peak in the same run").
// Every thread runs kChains independent dependent-FMA chains held in registers; nothing touches memory until the
// final store, so the kernel's duration is the FMA pipe's.  variant 0: scalar FFMA (three register operands);
// variant 1: packed FFMA2 (fma.rn.f32x2, two FMAs per lane per instruction -- the form the property kernels use).
#include "common.cuh"

namespace {

constexpr int kChains = 8;
constexpr int kProbeThreads = 256;

template <bool PACKED>
__global__ void __launch_bounds__(kProbeThreads)
fma_peak_kernel(long long iters, float a0, float b0, float* __restrict__ out) {
    const float seed = (float)threadIdx.x * 1e-3f;
    float r = 0.f;
    if (PACKED) {
        float2 x[kChains];
#pragma unroll
        for (int c = 0; c < kChains; ++c) x[c] = make_float2(seed + c, seed - c);
        const float2 a = make_float2(a0, a0), b = make_float2(b0, b0);
        for (long long i = 0; i < iters; ++i) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) x[c] = __ffma2_rn(x[c], a, b);
        }
#pragma unroll
        for (int c = 0; c < kChains; ++c) r += x[c].x + x[c].y;
    } else {
        float x[2 * kChains];
#pragma unroll
        for (int c = 0; c < 2 * kChains; ++c) x[c] = seed + c;
        for (long long i = 0; i < iters; ++i) {
#pragma unroll
            for (int c = 0; c < 2 * kChains; ++c) x[c] = fmaf(x[c], a0, b0);
        }
#pragma unroll
        for (int c = 0; c < 2 * kChains; ++c) r += x[c];
    }
    if (out) out[(size_t)blockIdx.x * kProbeThreads + threadIdx.x] = r;
}

// Issue rates behind the property kernels' pair loops: MODE 2 = eight independent chains of
// MUFU.RCP per iteration (each followed by an FADD so that rcp(rcp(x)) cannot be folded; the FADDs run on the FMA pipe, 1 clock
// each against the XU pipe's 8); MODE 3 = the pair loop's mix, 2 MUFU.RCP + 6 FFMA2 per iteration on eight independent chains.
template <int MODE>
__global__ void __launch_bounds__(128)
issue_probe_kernel(long long iters, float a0, float b0, float* __restrict__ out) {
    float r[8];
    float2 x[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        r[c] = 1.0f + (float)threadIdx.x * 1e-3f + c;
        x[c] = make_float2(r[c], r[c] + 1.f);
    }
    const float2 a = make_float2(a0, a0), b = make_float2(b0, b0);
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if (MODE == 2) {
                asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(r[c]));
                r[c] += 1.0f;
            } else {
                if (c < 2) {
                    asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(r[c]));
                    r[c] += 1.0f;
                }
                if (c < 6) x[c] = __ffma2_rn(x[c], a, b);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c) s += r[c] + x[c].x + x[c].y;
    if (out) out[(size_t)blockIdx.x * 128 + threadIdx.x] = s;
}

}  // namespace

extern "C" df_status df_probe_fp32_peak(int variant, int blocks, long long iters, float* out, double* flops, void* stream) {
    if (variant < 0 || variant > 3 || blocks < 1 || iters < 1)
        return df_set_error(DF_ERR_INVALID_ARG, "df_probe_fp32_peak: bad argument");
    if (variant >= 2) {   // issue-rate probes: blocks x 128 threads; *flops = warp-iterations of the launch
        if (variant == 2) issue_probe_kernel<2><<<blocks, 128, 0, (cudaStream_t)stream>>>(iters, 0.5f, 1.0f, out);
        else issue_probe_kernel<3><<<blocks, 128, 0, (cudaStream_t)stream>>>(iters, 0.5f, 1.0f, out);
        DF_CUDA_TRY(cudaGetLastError());
        if (flops) *flops = (double)iters * (double)blocks * 4.0;
        return DF_OK;
    }
    // out (optional) holds blocks * 256 floats; a, b keep the chains bounded (x -> 0.5 x + 1)
    if (variant == 1) fma_peak_kernel<true><<<blocks, kProbeThreads, 0, (cudaStream_t)stream>>>(iters, 0.5f, 1.0f, out);
    else fma_peak_kernel<false><<<blocks, kProbeThreads, 0, (cudaStream_t)stream>>>(iters, 0.5f, 1.0f, out);
    DF_CUDA_TRY(cudaGetLastError());
    if (flops) *flops = 2.0 * 2.0 * kChains * (double)iters * (double)blocks * kProbeThreads;   // both variants: 16 FMAs / thread / iteration
    return DF_OK;
}

// ann_fp32.cu -- K3: the ANN source term on the fp32 FFMA path (precision 0; BASELINE config 1,
// 11 -> 64 -> 64 -> 9).  Tensor cores cannot meet the 1e-5 tolerance of this path, so it is plain
// FFMA: one thread per cell, activations ping-pong through shared memory ([feature][thread],
// conflict-free), weights W^T[in][out] read warp-uniformly through the read-only path as float4,
// 8 outputs register-blocked per pass over the inputs.  Exact erf GELU (A13).
#include "ann_common.cuh"

namespace {

constexpr int kThreads = 64;
constexpr int kMaxLayers = 8;

struct Fp32Net {
    int n_layers;
    int dims[kMaxLayers + 1];
    int out_pad[kMaxLayers];
    const float* WT[kMaxLayers];  // [in][out_pad]
    const float* b[kMaxLayers];   // [out_pad]
    int max_dim;
};

__global__ void __launch_bounds__(kThreads)
ann_fp32_kernel(Fp32Net net, AnnNorm nm, int K, const float* __restrict__ invW, long long n, long long ld,
                const float* __restrict__ Tg, const float* __restrict__ pg, const float* __restrict__ Yg,
                float* __restrict__ omega, float* __restrict__ dY) {
    extern __shared__ float sm[];
    const int t = threadIdx.x;
    float* act0 = sm;
    float* act1 = sm + (size_t)net.max_dim * kThreads;
    const long long i = (long long)blockIdx.x * kThreads + t;
    if (i >= n) return;

    const float T = __ldg(Tg + i), p = __ldg(pg + i);
    act0[0 * kThreads + t] = (T - nm.x_mean[0]) * nm.x_inv_std[0];
    act0[1 * kThreads + t] = (p - nm.x_mean[1]) * nm.x_inv_std[1];
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        act0[(2 + k) * kThreads + t] = ann_feature_Y(y, nm.lambda, nm.inv_lambda, nm.x_mean[2 + k], nm.x_inv_std[2 + k]);
    }

    float* in = act0;
    float* out = act1;
    for (int l = 0; l < net.n_layers; ++l) {
        const int din = net.dims[l], dout = net.dims[l + 1], op = net.out_pad[l];
        const bool last = (l + 1 == net.n_layers);
        for (int o = 0; o < dout; o += 8) {
            float acc[8];
            const float4 b0 = __ldg(reinterpret_cast<const float4*>(net.b[l] + o));
            const float4 b1 = __ldg(reinterpret_cast<const float4*>(net.b[l] + o + 4));
            acc[0] = b0.x; acc[1] = b0.y; acc[2] = b0.z; acc[3] = b0.w;
            acc[4] = b1.x; acc[5] = b1.y; acc[6] = b1.z; acc[7] = b1.w;
            const float* w = net.WT[l] + o;
#pragma unroll 4
            for (int ii = 0; ii < din; ++ii) {
                const float a = in[ii * kThreads + t];
                const float4 w0 = __ldg(reinterpret_cast<const float4*>(w + (size_t)ii * op));
                const float4 w1 = __ldg(reinterpret_cast<const float4*>(w + (size_t)ii * op + 4));
                acc[0] = fmaf(a, w0.x, acc[0]); acc[1] = fmaf(a, w0.y, acc[1]);
                acc[2] = fmaf(a, w0.z, acc[2]); acc[3] = fmaf(a, w0.w, acc[3]);
                acc[4] = fmaf(a, w1.x, acc[4]); acc[5] = fmaf(a, w1.y, acc[5]);
                acc[6] = fmaf(a, w1.z, acc[6]); acc[7] = fmaf(a, w1.w, acc[7]);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (o + j < dout) out[(o + j) * kThreads + t] = last ? acc[j] : gelu_erf(acc[j]);
        }
        float* tmp = in; in = out; out = tmp;
    }
    // `in` now holds the K network outputs o_k; `out` is scratch for dY*_k.
    double sumYm1 = -1.0, sumd = 0.0;
    float inv_Wbar = 0.f;
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        const float delta = fmaf(nm.u_std[k], in[k * kThreads + t], nm.u_mean[k]);
        const float d = ann_dystar(y, delta, nm.lambda, nm.inv_lambda);
        out[k * kThreads + t] = d;
        sumYm1 += (double)y;
        sumd += (double)d;
        inv_Wbar = fmaf(y, __ldg(invW + k), inv_Wbar);
    }
    const double Sm1 = sumYm1 + sumd;
    const double inv_S = 1.0 / (1.0 + Sm1);
    const float rho_dt = p / (inv_Wbar * (float)DF_R_UNIVERSAL * T) * nm.inv_dt;  // A17
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        const float d = ann_renorm_dY(out[k * kThreads + t], y, Sm1, inv_S);
        if (dY) dY[(size_t)k * ld + i] = d;
        if (omega) omega[(size_t)k * ld + i] = rho_dt * d;
    }
}

}  // namespace

df_status launch_ann_fp32(const df_ann* ann, const df_mech* mech, long long n, long long ld, const float* T,
                          const float* p, const float* Y, float* omega, float* dY, cudaStream_t s) {
    Fp32Net net;
    net.n_layers = ann->n_layers;
    net.max_dim = 0;
    for (int l = 0; l <= ann->n_layers; ++l) {
        net.dims[l] = ann->dims[l];
        if (ann->dims[l] > net.max_dim) net.max_dim = ann->dims[l];
    }
    for (int l = 0; l < ann->n_layers; ++l) {
        net.out_pad[l] = ann->out_pad[l];
        net.WT[l] = ann->w32 + ann->w32_off[l];
        net.b[l] = ann->w32 + ann->b32_off[l];
    }
    const size_t smem = (size_t)2 * net.max_dim * kThreads * sizeof(float);
    static DfPerDevice smem_attr;
    const df_status st = df_ensure_dyn_smem((const void*)ann_fp32_kernel, 200 * 1024, &smem_attr);
    if (st != DF_OK) return st;
    const long long blocks = (n + kThreads - 1) / kThreads;
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_chem_ann_source: n_cells too large");
    ann_fp32_kernel<<<(unsigned)blocks, kThreads, smem, s>>>(net, ann->norm, ann->K, mech->dev.invW, n, ld, T, p, Y,
                                                            omega, dY);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

// ann_fp32.cu -- K3: the ANN source term on the fp32 FFMA path (precision 0; BASELINE config 1,
// 11 -> 64 -> 64 -> 9).  Tensor cores cannot meet the 1e-5 tolerance of this path, so it is plain
// FFMA.  A block owns 32 cells; lane = cell, and the eight warps split every layer's outputs (warp j takes outputs
// 8j .. 8j+7, then +64, ...: a cell's serial chain is an eighth of the layer), activations ping-pong through shared
// memory ([feature][cell], conflict-free), weights W^T[in][out] are fetched a layer ahead into shared memory with cp.async
// (all loads of a layer in flight at once; read from global memory each one was an L2 round trip on the chain: 36 -> 15 us)
// and read warp-uniformly as float4.  Exact erf GELU (A13).  The configuration is launch/latency-bound (4096 cells), so what counts is the length
// of the per-cell dependency chain, not throughput.
#include "ann_common.cuh"

namespace {

constexpr int kCells = 32;               // cells per block (one per lane)
constexpr int kSplit = 8;                // warps per block = output slices
constexpr int kThreads = kCells * kSplit;
constexpr int kMaxLayers = 8;

struct Fp32Net {
    int n_layers;
    int dims[kMaxLayers + 1];
    int out_pad[kMaxLayers];
    const float* WT[kMaxLayers];  // [in][out_pad]
    const float* b[kMaxLayers];   // [out_pad]
    int max_dim;
    int stage_floats;   // > 0: every layer's W^T and bias fit a shared-memory buffer of this many floats (two of them: double-buffered)
};

__global__ void __launch_bounds__(kThreads)
ann_fp32_kernel(Fp32Net net, AnnNorm nm, int K, const float* __restrict__ invW, long long n, long long ld,
                const float* __restrict__ Tg, const float* __restrict__ pg, const float* __restrict__ Yg,
                float* __restrict__ omega, float* __restrict__ dY) {
    extern __shared__ float sm[];
    const int c = threadIdx.x & 31, j = threadIdx.x >> 5;
    float* act0 = sm;
    float* act1 = sm + (size_t)net.max_dim * kCells;
    float* wbuf = act1 + (size_t)net.max_dim * kCells;   // 2 x stage_floats: layer l's W^T then its bias, staged with cp.async
    // A weight is read once per block, so from global memory every read is an L2 round trip on the cell's dependency chain;
    // the whole layer is fetched with all loads in flight at once instead, one layer ahead of its use.
    auto stage = [&](int l) {
        if (net.stage_floats == 0 || l >= net.n_layers) return;
        float* dst = wbuf + (size_t)(l & 1) * net.stage_floats;
        const int nw = net.dims[l] * net.out_pad[l], nb = net.out_pad[l];
        for (int e = threadIdx.x * 4; e < nw; e += kThreads * 4)
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst + e)), "l"(net.WT[l] + e) : "memory");
        for (int e = threadIdx.x * 4; e < nb; e += kThreads * 4)
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst + nw + e)), "l"(net.b[l] + e) : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    stage(0);
    const long long i_raw = (long long)blockIdx.x * kCells + c;
    const bool valid = i_raw < n;
    const long long i = valid ? i_raw : 0;   // every thread stays for the barriers; cells past the end are not stored

    const float T = __ldg(Tg + i), p = __ldg(pg + i);
    for (int f = j; f < K + 2; f += kSplit) {
        float x;
        if (f == 0) x = (T - nm.x_mean[0]) * nm.x_inv_std[0];
        else if (f == 1) x = (p - nm.x_mean[1]) * nm.x_inv_std[1];
        else x = ann_feature_Y(__ldg(Yg + (size_t)(f - 2) * ld + i), nm.lambda, nm.inv_lambda, nm.x_mean[f], nm.x_inv_std[f]);
        act0[f * kCells + c] = x;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();

    float* in = act0;
    float* out = act1;
    for (int l = 0; l < net.n_layers; ++l) {
        const int din = net.dims[l], dout = net.dims[l + 1], op = net.out_pad[l];
        const bool last = (l + 1 == net.n_layers);
        stage(l + 1);
        const bool staged = net.stage_floats > 0;
        const float* wl = staged ? wbuf + (size_t)(l & 1) * net.stage_floats : net.WT[l];
        const float* bl = staged ? wl + din * op : net.b[l];
        for (int o = j * 8; o < dout; o += 8 * kSplit) {
            float acc[8];
            const float4 b0 = *reinterpret_cast<const float4*>(bl + o);
            const float4 b1 = *reinterpret_cast<const float4*>(bl + o + 4);
            acc[0] = b0.x; acc[1] = b0.y; acc[2] = b0.z; acc[3] = b0.w;
            acc[4] = b1.x; acc[5] = b1.y; acc[6] = b1.z; acc[7] = b1.w;
            const float* w = wl + o;
#pragma unroll 4
            for (int ii = 0; ii < din; ++ii) {
                const float a = in[ii * kCells + c];
                const float4 w0 = *reinterpret_cast<const float4*>(w + (size_t)ii * op);
                const float4 w1 = *reinterpret_cast<const float4*>(w + (size_t)ii * op + 4);
                acc[0] = fmaf(a, w0.x, acc[0]); acc[1] = fmaf(a, w0.y, acc[1]);
                acc[2] = fmaf(a, w0.z, acc[2]); acc[3] = fmaf(a, w0.w, acc[3]);
                acc[4] = fmaf(a, w1.x, acc[4]); acc[5] = fmaf(a, w1.y, acc[5]);
                acc[6] = fmaf(a, w1.z, acc[6]); acc[7] = fmaf(a, w1.w, acc[7]);
            }
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (o + q < dout) out[(o + q) * kCells + c] = last ? acc[q] : gelu_erf(acc[q]);
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
        float* tmp = in; in = out; out = tmp;
    }
    // `in` now holds the K network outputs o_k; `out` is scratch for dY*_k (species k = j, j + 8, ... per warp).
    for (int k = j; k < K; k += kSplit) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        const float delta = fmaf(nm.u_std[k], in[k * kCells + c], nm.u_mean[k]);
        out[k * kCells + c] = ann_dystar(y, delta, nm.lambda, nm.inv_lambda);
    }
    __syncthreads();
    // every warp forms the two sums in the same order (bitwise identical in all of them), then finishes its species
    double sumYm1 = -1.0, sumd = 0.0;
    float inv_Wbar = 0.f;
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        sumYm1 += (double)y;
        sumd += (double)out[k * kCells + c];
        inv_Wbar = fmaf(y, __ldg(invW + k), inv_Wbar);
    }
    const double Sm1 = sumYm1 + sumd;
    const double inv_S = 1.0 / (1.0 + Sm1);
    const float rho_dt = p / (inv_Wbar * (float)DF_R_UNIVERSAL * T) * nm.inv_dt;  // A17
    if (valid)
        for (int k = j; k < K; k += kSplit) {
            const float y = __ldg(Yg + (size_t)k * ld + i);
            const float d = ann_renorm_dY(out[k * kCells + c], y, Sm1, inv_S);
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
    // stage the weights in shared memory when every layer (W^T + bias) fits 16 K floats and is 16-byte aligned
    int stage_floats = 0;
    bool can_stage = true;
    for (int l = 0; l < ann->n_layers; ++l) {
        const int fl = ann->dims[l] * ann->out_pad[l] + ann->out_pad[l];
        if (fl > stage_floats) stage_floats = fl;
        if (ann->w32_off[l] % 4 || ann->b32_off[l] % 4 || ann->out_pad[l] % 4) can_stage = false;
    }
    if (!can_stage || stage_floats > 16384) stage_floats = 0;
    stage_floats = (stage_floats + 3) / 4 * 4;
    net.stage_floats = stage_floats;
    const size_t smem = ((size_t)2 * net.max_dim * kCells + (size_t)2 * stage_floats) * sizeof(float);
    static DfPerDevice smem_attr;
    const df_status st = df_ensure_dyn_smem((const void*)ann_fp32_kernel, 200 * 1024, &smem_attr);
    if (st != DF_OK) return st;
    const long long blocks = (n + kCells - 1) / kCells;
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_chem_ann_source: n_cells too large");
    ann_fp32_kernel<<<(unsigned)blocks, kThreads, smem, s>>>(net, ann->norm, ann->K, mech->dev.invW, n, ld, T, p, Y,
                                                            omega, dY);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

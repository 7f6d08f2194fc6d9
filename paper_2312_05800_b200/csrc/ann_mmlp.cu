// ann_mmlp.cu -- NEXT-1: one MLP per species ("individual training and prediction ... for each species mass
// fraction"; "multiple multilayer perceptrons"): K independent networks (K+2) -> d1 -> d2 -> d3 -> 1 on the
// tensor path.  Each network is the tcgen05 chain of ann_bf16.cu, launched once per species on the caller's stream
// with its last layer embedded as row k of a K-row matrix (the other rows are zero), in "raw" mode: its final epilogue
// stores o_k = a_3 . w_k + b_k to row k of a scratch array instead of running the inverse transform.  One pointwise
// kernel then applies the shared epilogue (A9-A11, A17) to the K outputs of a cell.  The prologue (21 features) is
// recomputed by every launch -- it runs on the I/O warps, off the MMA critical path -- and the o_k round trip through
// HBM is 4 K bytes per cell against 62 MFLOP per cell of tensor work.
#include <cstring>
#include <new>

#include "ann_common.cuh"

struct df_ann_mmlp {
    int K;
    std::vector<df_ann*> nets;   // K handles of the single-network path, each with a one-row last layer
    AnnNorm norm;                // shared x statistics, per-species u statistics, lambda, dt
};

namespace {

constexpr int kET = 128;

// epilogue of P:79 / A9-A11, A17 on the K raw outputs of a cell (same arithmetic as the fp32 path: expm1/log1p form,
// fp64 sums)
__global__ void __launch_bounds__(kET)
mmlp_epilogue_kernel(AnnNorm nm, int K, const float* __restrict__ invW, long long n, long long ld, const float* __restrict__ raw,
                     const float* __restrict__ Tg, const float* __restrict__ pg, const float* __restrict__ Yg,
                     float* __restrict__ omega, float* __restrict__ dY) {
    const long long i = (long long)blockIdx.x * kET + threadIdx.x;
    if (i >= n) return;
    const float T = __ldg(Tg + i), p = __ldg(pg + i);
    double sumYm1 = -1.0, sumd = 0.0;
    float inv_Wbar = 0.f;
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        const float delta = fmaf(nm.u_std[k], __ldg(raw + (size_t)k * ld + i), nm.u_mean[k]);
        sumYm1 += (double)y;
        sumd += (double)ann_dystar(y, delta, nm.lambda, nm.inv_lambda);
        inv_Wbar = fmaf(y, __ldg(invW + k), inv_Wbar);
    }
    const double Sm1 = sumYm1 + sumd, inv_S = 1.0 / (1.0 + Sm1);
    const float rho_dt = p / (inv_Wbar * (float)DF_R_UNIVERSAL * T) * nm.inv_dt;
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        const float delta = fmaf(nm.u_std[k], __ldg(raw + (size_t)k * ld + i), nm.u_mean[k]);
        const float d = ann_renorm_dY(ann_dystar(y, delta, nm.lambda, nm.inv_lambda), y, Sm1, inv_S);
        if (dY) dY[(size_t)k * ld + i] = d;
        if (omega) omega[(size_t)k * ld + i] = rho_dt * d;
    }
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
size_t raw_bytes(int K, long long ld) { return ((size_t)K * (size_t)ld * sizeof(float) + 1023) / 1024 * 1024; }

}  // namespace

extern "C" df_status df_ann_mmlp_destroy(df_ann_mmlp* m) {
    if (!m) return DF_OK;
    for (df_ann* a : m->nets) df_ann_destroy(a);
    delete m;
    return DF_OK;
}

extern "C" df_status df_ann_mmlp_create(df_ann_mmlp** out, int K, int n_layers, const int* dims, const float* const* W,
                                        const float* const* b, const double* x_mean, const double* x_std,
                                        const double* u_mean, const double* u_std, double boxcox_lambda, double dt) {
    if (!out) return df_set_error(DF_ERR_INVALID_ARG, "df_ann_mmlp_create: out is NULL");
    *out = nullptr;
    if (!dims || !W || !b || !x_mean || !x_std || !u_mean || !u_std)
        return df_set_error(DF_ERR_INVALID_ARG, "df_ann_mmlp_create: NULL argument");
    if (n_layers != 4) return df_set_error(DF_ERR_UNSUPPORTED, "df_ann_mmlp_create: the tensor path takes n_layers = 4 (got %d)", n_layers);
    if (K < 1 || K > 28 || dims[0] != K + 2 || dims[4] != 1)
        return df_set_error(DF_ERR_INVALID_ARG, "df_ann_mmlp_create: need dims[0] == K + 2, dims[4] == 1, K <= 28");
    df_ann_mmlp* m = new (std::nothrow) df_ann_mmlp;
    if (!m) return df_set_error(DF_ERR_ALLOC, "df_ann_mmlp_create: out of host memory");
    m->K = K;
    const int d3 = dims[3];
    int dims_k[5] = {dims[0], dims[1], dims[2], dims[3], K};
    std::vector<float> W4((size_t)K * d3), b4(K);
    for (int k = 0; k < K; ++k) {
        for (int l = 0; l < 4; ++l)
            if (!W[k * 4 + l] || !b[k * 4 + l]) {
                df_ann_mmlp_destroy(m);
                return df_set_error(DF_ERR_INVALID_ARG, "df_ann_mmlp_create: net %d layer %d is NULL", k, l);
            }
        // the one-row last layer of net k as row k of a K-row matrix (zeros are bf16-valued)
        std::fill(W4.begin(), W4.end(), 0.f);
        std::fill(b4.begin(), b4.end(), 0.f);
        memcpy(&W4[(size_t)k * d3], W[k * 4 + 3], sizeof(float) * d3);
        b4[k] = b[k * 4 + 3][0];
        const float* Wk[4] = {W[k * 4], W[k * 4 + 1], W[k * 4 + 2], W4.data()};
        const float* bk[4] = {b[k * 4], b[k * 4 + 1], b[k * 4 + 2], b4.data()};
        df_ann* a = nullptr;
        const df_status st = df_ann_create(&a, 4, dims_k, Wk, bk, 1, x_mean, x_std, u_mean, u_std, boxcox_lambda, dt);
        if (st != DF_OK) {
            df_ann_mmlp_destroy(m);
            return st;
        }
        m->nets.push_back(a);
    }
    m->norm = m->nets[0]->norm;
    *out = m;
    return DF_OK;
}

extern "C" size_t df_ann_mmlp_workspace_bytes(const df_ann_mmlp* m, long long n_cells, long long ld) {
    if (!m || n_cells <= 0 || ld < n_cells) return 0;
    return raw_bytes(m->K, ld) + ann_bf16_workspace(m->nets[0], n_cells);
}

extern "C" df_status df_chem_ann_source_mmlp(const df_ann_mmlp* m, const df_mech* mech, long long n, long long ld,
                                             const float* T, const float* p, const float* Y, float* omega, float* dY,
                                             void* workspace, size_t workspace_bytes, void* stream) {
    if (!m || !mech) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: NULL handle");
    if (m->K != mech->K) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: nets have K=%d, mech has K=%d", m->K, mech->K);
    if (n < 0 || ld < n || ld % 4 != 0) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: bad n_cells / ld");
    if (n == 0) return DF_OK;
    if (!T || !p || !Y) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: NULL input field");
    if (!omega && !dY) return DF_OK;
    if (!aligned16(T) || !aligned16(p) || !aligned16(Y) || !aligned16(omega) || !aligned16(dY))
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: fields must be 16-byte aligned");
    const size_t rb = raw_bytes(m->K, ld), sb = ann_bf16_workspace(m->nets[0], n);
    if (!workspace || workspace_bytes < rb + sb)
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: workspace of %zu bytes needed, %zu given", rb + sb,
                            workspace ? workspace_bytes : (size_t)0);
    if (reinterpret_cast<uintptr_t>(workspace) & 1023u)
        return df_set_error(DF_ERR_INVALID_ARG, "df_chem_ann_source_mmlp: workspace must be 1024-byte aligned");
    if ((n + kET - 1) / kET > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_chem_ann_source_mmlp: n_cells too large");
    float* raw = static_cast<float*>(workspace);
    void* scratch = static_cast<uint8_t*>(workspace) + rb;
    for (int k = 0; k < m->K; ++k) {
        const df_status st = launch_ann_bf16(m->nets[k], mech, n, ld, T, p, Y, nullptr, nullptr, scratch, sb, (cudaStream_t)stream, raw, k);
        if (st != DF_OK) return st;
    }
    mmlp_epilogue_kernel<<<(unsigned)((n + kET - 1) / kET), kET, 0, (cudaStream_t)stream>>>(m->norm, m->K, mech->dev.invW, n, ld, raw, T, p, Y,
                                                                                            omega, dY);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

// common.cuh -- handle layouts and small device helpers shared by the libdfthermo.so sources.
// Product code: nothing here is used by, or uses, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <vector>

#include "../../include/df_thermo.h"

#define DF_MAX_K 64
#define DF_R_UNIVERSAL 8314.46261815324

// ---- error plumbing ---------------------------------------------------------------------------
df_status df_set_error(df_status code, const char* fmt, ...);
#define DF_CUDA_TRY(expr)                                                                         \
    do {                                                                                          \
        cudaError_t e__ = (expr);                                                                 \
        if (e__ != cudaSuccess)                                                                   \
            return df_set_error(DF_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), \
                                __FILE__, __LINE__);                                              \
    } while (0)

// ---- per-device launch prerequisites (runtime.cu) ------------------------------------------------
// cudaFuncSetAttribute applies to the device that is current when it is called, so "done once" must be tracked per
// device, not per process (a second GPU in the same process would otherwise launch without the attribute).
struct DfPerDevice {
    std::atomic<unsigned long long> done[2] = {{0ull}, {0ull}};   // one bit per device ordinal (up to 128)
};
df_status df_ensure_dyn_smem(const void* kernel, int bytes, DfPerDevice* state);
int df_device_sm_count();   // multiprocessors of the current device (cached per device); 0 on error

// ---- species tables, repacked at create time (mech.cu) ---------------------------------------
// Thermo: h_k(T)/W_k = sum_{m<6} th[k][r][m] tau^m with tau = (T - T_mid) * inv_S, r = 0 (lo) / 1 (hi).
// Transport: u = (ln T - Lc) * inv_Ls; ghat_k = sqrt(mu_k)/(T W_k)^(1/4) = sum_m visc[k][m] u^m;
// lambda_k/sqrt(T) = sum_m cond[k][m] u^m; p D_jk / T^(3/2) = sum_m dpair[..][m] u^m.
struct MechScalars {
    float T_mid, inv_S, S, Lc, inv_Ls;
    float tau_min, tau_max;  // Newton clamp [50 K, 6000 K] in tau
};

// Generic-K device tables (global memory; kernels stage what they need into shared memory).
constexpr int kWilkeRank = 12;
struct MechDev {
    int K;
    MechScalars sc;
    float* th32;     // [K][2][6]
    float* sth32;    // [K][2][6]  s_k(T)/W_k = sth[0] ln T + sum_{m<5} sth[1+m] tau^m   (pointwise.cu)
    double* th64;    // [K][2][6]
    float* invW;     // [K]
    float* sqrtW;    // [K]
    float* visc;     // [K][5]   (W_k^(-1/4) folded in)
    float* cond;     // [K][5]
    float* ddiag;    // [K][5]
    float* dfull;    // [K][K][5] symmetric, generic path
    float* wilkeB;   // [K][K]   B_kj = 1/sqrt(8 (1 + W_k/W_j))
    // padded / tiled copies for the any-K kernel (properties_group.cu); Kp = K rounded up to 8, nt = Kp / 8
    int Kp;
    float* small_p;  // [Kp][20]: invW, sqrtW, visc[5], cond[5], ddiag[5], pad(3); padding species: visc = cond = ddiag = 1, rest 0
    float* thp;      // [Kp][2][6] fp32 thermo (padding: 0)
    double* h0p;     // [Kp][2]   fp64 constant terms
    float* BW;       // [4][Kp][16]: BW[w][j][a] = B_{k,j} for k = w Kp/4 + a (Wilke rows of warp w; padding 1)
    // Wilke's B in factored form (properties_group.cu, K > 28): B = U diag(s) V^T truncated after wilke_rank = 8 or 12 terms -- B depends
    // on W_k/W_j only and is smooth in it, so its singular values fall by ~10x per term.  wilke_rank = 0: not usable (the
    // truncation error of this mechanism's B exceeds 1e-6 element-wise -- a tenth of the 1e-5 tolerance of mu --, or K is too small to gain) -> the full table BW is used.
    int wilke_rank;
    float* VW;       // [4][Kp][4]:  VW[w][j][c] = V_{j, w + 4c} (modes of warp w; c = 3 and padding species: 0)
    float* UW;       // [4][kWilkeRank][16] (wilke_rank rows used): UW[w][m][a] = U_{k,m} s_m for k = w Kp/4 + a (padding rows: 1 for m = 0, else 0)
    float* dtile;    // eight species tiles of TS = Kp/8: [36 tile pairs (kt <= jt)][TS][row of TS x 5, padded to 4 floats]
                     // = coefficients of D_{kt TS + a, jt TS + b} (padding pairs: 1,0,0,0,0)
};

// Fixed-K tables passed as a __grid_constant__ kernel parameter: every coefficient becomes a
// constant-bank operand of the FFMA that consumes it (no load instruction in the inner loops).
template <int K>
struct PropTables {
    double h0[K][2];
    float th[K][2][5];  // m = 1..5
    float invW[K], sqrtW[K];
    float visc[K][5], cond[K][5], ddiag[K][5];
    float B[K][K];
    // Wilke's B factored, B_kj ~ sum_{m < wilke_rank} WU[k][m] WV[j][m] (WU carries the singular values); wilke_rank = 0: use B
    float WV[K][8], WU[K][8];
    int wilke_rank;
    float dpair[K * (K - 1) / 2 > 0 ? K * (K - 1) / 2 : 1][5];  // pairs (j<k) in row-major order of (j,k)
    MechScalars sc;
};

struct df_mech {
    int K;
    MechDev dev;
    std::vector<double> W_host;
    std::vector<double> th64_host;  // [K][2][6] host copy of dev.th64 (fixed-K Newton tables are built from it per launch)
    PropTables<9>* t9 = nullptr;    // host copies of the fixed-K tables (only the matching one is set)
    PropTables<19>* t19 = nullptr;
};

// ---- ANN tables --------------------------------------------------------------------------------
struct AnnNorm {                 // passed by value to kernels (K <= 64)
    float x_mean[DF_MAX_K + 2], x_inv_std[DF_MAX_K + 2];
    float u_mean[DF_MAX_K], u_std[DF_MAX_K];
    float lambda, inv_lambda, inv_dt;
};

struct Bf16Plan;  // ann_bf16.cu

struct df_ann {
    int n_layers;
    std::vector<int> dims;
    int precision;
    int K;
    AnnNorm norm;
    // fp32 path: per layer W^T [in][out_pad4] and b [out_pad4], one device allocation
    float* w32 = nullptr;
    std::vector<size_t> w32_off, b32_off;
    std::vector<int> out_pad;
    Bf16Plan* bf16 = nullptr;
};

// ---- device helpers ----------------------------------------------------------------------------
__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float poly4(const float* c, float u) {
    return fmaf(fmaf(fmaf(fmaf(c[4], u, c[3]), u, c[2]), u, c[1]), u, c[0]);
}

// launchers implemented in the kernel translation units
df_status launch_T_from_h(const df_mech*, long long n, long long ld, const float* h, const float* Y, float* T,
                          float* cp, int* n_unconv, cudaStream_t s);
df_status launch_properties_group(const df_mech*, long long n, long long ld, const float* T, const float* p, const float* Y,
                                  float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s);
df_status launch_properties(const df_mech*, long long n, long long ld, const float* T, const float* p, const float* Y,
                            float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s);
df_status launch_ann_fp32(const df_ann*, const df_mech*, long long n, long long ld, const float* T, const float* p,
                          const float* Y, float* omega, float* dY, cudaStream_t s);
df_status ann_bf16_create(df_ann*, const float* const* W, const float* const* b);
void ann_bf16_destroy(df_ann*);
size_t ann_bf16_workspace(const df_ann*, long long n);
df_status launch_ann_bf16(const df_ann*, const df_mech*, long long n, long long ld, const float* T, const float* p,
                          const float* Y, float* omega, float* dY, void* ws, size_t ws_bytes, cudaStream_t s,
                          float* raw = nullptr, int raw_row = 0);

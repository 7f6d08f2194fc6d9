// properties.cu -- K2: fused mixture thermo + transport pass (NS (2)).
//
// FP32-FMA-bound for every K (12.5 K^2 + 51.5 K flops per cell against 4(2K+6) bytes), so the
// design goal is FMA density, not bytes:
//   * fixed-K kernels (K = 9, 19) take the whole species table as a __grid_constant__ parameter:
//     fully unrolled, every coefficient is a constant-bank operand of its FFMA (no loads in the
//     inner loops), all per-cell vectors live in registers;
//   * Wilke's sum is evaluated in its three-vector form, 3 FFMA per (k,j):
//       sum_j X_j Phi_kj = sum_j B_kj (X_j + g_k (2 X_j/g_j + g_k X_j/g_j^2)),  g = sqrt(mu)/(T W)^(1/4);
//   * binary diffusion uses each symmetric pair once (4 FFMA Horner + 1 MUFU.RCP + 2 FFMA);
//   * the formation-enthalpy part of h is accumulated in fp64 (K DFMA), the sensible part in fp32.
// A generic-K kernel (any K <= 64, per-thread vectors in shared memory) covers the other sizes.
#include "common.cuh"

namespace {

constexpr int kThreads = 128;

// ------------------------------------------------------------------------------------------------
// fixed K
// ------------------------------------------------------------------------------------------------
template <int K, bool TRANSPORT>
__global__ void __launch_bounds__(kThreads)
props_fixed_kernel(const __grid_constant__ PropTables<K> tab, long long n, long long ld,
                   const float* __restrict__ Tg, const float* __restrict__ pg, const float* __restrict__ Yg,
                   float* __restrict__ cp_o, float* __restrict__ h_o, float* __restrict__ mu_o,
                   float* __restrict__ lam_o, float* __restrict__ D_o) {
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i >= n) return;
    const float T = __ldg(Tg + i);
    float Y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) Y[k] = __ldg(Yg + (size_t)k * ld + i);

    // ---- thermo: mixture polynomial in tau, both ranges, select at the end ---------------------
    const float tau = (T - tab.sc.T_mid) * tab.sc.inv_S;
    const bool lo = T < tab.sc.T_mid;  // A2: hi for T >= T_mid
    if (cp_o || h_o) {
        float Cl[5] = {0.f, 0.f, 0.f, 0.f, 0.f}, Ch[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
        double H0l = 0.0, H0h = 0.0;
#pragma unroll
        for (int k = 0; k < K; ++k) {
#pragma unroll
            for (int m = 0; m < 5; ++m) {
                Cl[m] = fmaf(Y[k], tab.th[k][0][m], Cl[m]);
                Ch[m] = fmaf(Y[k], tab.th[k][1][m], Ch[m]);
            }
            const double yd = (double)Y[k];
            H0l = fma(yd, tab.h0[k][0], H0l);
            H0h = fma(yd, tab.h0[k][1], H0h);
        }
        float q[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = lo ? Cl[m] : Ch[m];
        const float sens = tau * fmaf(fmaf(fmaf(fmaf(q[4], tau, q[3]), tau, q[2]), tau, q[1]), tau, q[0]);
        if (h_o) h_o[i] = (float)((lo ? H0l : H0h) + (double)sens);
        if (cp_o)
            cp_o[i] = fmaf(fmaf(fmaf(fmaf(5.f * q[4], tau, 4.f * q[3]), tau, 3.f * q[2]), tau, 2.f * q[1]), tau, q[0]) *
                      tab.sc.inv_S;
    }
    if (!TRANSPORT) return;

    // ---- mole fractions -----------------------------------------------------------------------
    float X[K];
    float sumx = 0.f;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        X[k] = Y[k] * tab.invW[k];
        sumx += X[k];
    }
    const float inv_sumx = 1.0f / sumx;
#pragma unroll
    for (int k = 0; k < K; ++k) X[k] *= inv_sumx;

    const float u = (logf(T) - tab.sc.Lc) * tab.sc.inv_Ls;
    const float sqrtT = sqrtf(T);

    // ---- Wilke viscosity ----------------------------------------------------------------------
    if (mu_o) {
        float g[K], b2[K], c[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            g[k] = poly4(tab.visc[k], u);
            const float rg = rcp_approx(g[k]);
            const float xr = X[k] * rg;
            b2[k] = 2.f * xr;
            c[k] = xr * rg;
        }
        float acc = 0.f;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            float den = 0.f;
#pragma unroll
            for (int j = 0; j < K; ++j) den = fmaf(tab.B[k][j], fmaf(g[k], fmaf(g[k], c[j], b2[j]), X[j]), den);
            acc = fmaf(X[k] * tab.sqrtW[k] * g[k] * g[k], rcp_approx(den), acc);
        }
        mu_o[i] = sqrtT * acc;
    }

    // ---- combination-rule conductivity (A6) ---------------------------------------------------
    if (lam_o) {
        float s1 = 0.f, s2 = 0.f;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const float lk = poly4(tab.cond[k], u);
            s1 = fmaf(X[k], lk, s1);
            s2 = fmaf(X[k], rcp_approx(lk), s2);
        }
        lam_o[i] = 0.5f * sqrtT * (s1 + rcp_approx(s2));
    }

    // ---- mixture-averaged diffusivities (A7) ---------------------------------------------
    if (D_o) {
        const float p = __ldg(pg + i);
        const float scale = T * sqrtT / p;
        float S[K];
#pragma unroll
        for (int k = 0; k < K; ++k) S[k] = 0.f;
        {
            int idx = 0;
#pragma unroll
            for (int j = 0; j < K; ++j)
#pragma unroll
                for (int k = j + 1; k < K; ++k, ++idx) {
                    const float r = rcp_approx(poly4(tab.dpair[idx], u));
                    S[k] = fmaf(X[j], r, S[k]);
                    S[j] = fmaf(X[k], r, S[j]);
                }
        }
        // N_k = sum_{j != k} Y_j as prefix + suffix (never 1 - Y_k: cancels when Y_k -> 1)
        float suf[K + 1];
        suf[K] = 0.f;
#pragma unroll
        for (int k = K - 1; k >= 0; --k) suf[k] = suf[k + 1] + Y[k];
        float pre = 0.f;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const float Nk = pre + suf[k + 1];
            pre += Y[k];
            const float Dk = (S[k] > 0.f) ? Nk / S[k] : poly4(tab.ddiag[k], u);
            D_o[(size_t)k * ld + i] = Dk * scale;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// generic K (per-thread vectors in shared memory, tables through the read-only path)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads)
props_generic_kernel(MechDev md, long long n, long long ld, const float* __restrict__ Tg,
                     const float* __restrict__ pg, const float* __restrict__ Yg, float* __restrict__ cp_o,
                     float* __restrict__ h_o, float* __restrict__ mu_o, float* __restrict__ lam_o,
                     float* __restrict__ D_o) {
    extern __shared__ float sm[];
    const int K = md.K;
    const int t = threadIdx.x;
    float* sX = sm;                       // [K][kThreads]
    float* sG = sX + (size_t)K * kThreads;  // g_k
    float* sB = sG + (size_t)K * kThreads;  // 2 X/g
    float* sC = sB + (size_t)K * kThreads;  // X/g^2
    const long long i = (long long)blockIdx.x * kThreads + t;
    if (i >= n) return;
    const float T = __ldg(Tg + i);
    const float tau = (T - md.sc.T_mid) * md.sc.inv_S;
    const int r = (T < md.sc.T_mid) ? 0 : 1;

    float q[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
    double H0 = 0.0;
    float sumx = 0.f, sumY = 0.f;
    for (int k = 0; k < K; ++k) {
        const float y = __ldg(Yg + (size_t)k * ld + i);
        const float* c32 = md.th32 + (k * 2 + r) * 6;
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = fmaf(y, __ldg(c32 + 1 + m), q[m]);
        H0 = fma((double)y, __ldg(md.th64 + (k * 2 + r) * 6), H0);
        const float x = y * __ldg(md.invW + k);
        sX[k * kThreads + t] = x;
        sumx += x;
        sumY += y;
    }
    if (h_o) {
        const float sens = tau * fmaf(fmaf(fmaf(fmaf(q[4], tau, q[3]), tau, q[2]), tau, q[1]), tau, q[0]);
        h_o[i] = (float)(H0 + (double)sens);
    }
    if (cp_o)
        cp_o[i] = fmaf(fmaf(fmaf(fmaf(5.f * q[4], tau, 4.f * q[3]), tau, 3.f * q[2]), tau, 2.f * q[1]), tau, q[0]) *
                  md.sc.inv_S;
    if (!mu_o && !lam_o && !D_o) return;

    const float inv_sumx = 1.0f / sumx;
    const float u = (logf(T) - md.sc.Lc) * md.sc.inv_Ls;
    const float sqrtT = sqrtf(T);
    float s1 = 0.f, s2 = 0.f;
    for (int k = 0; k < K; ++k) {
        const float X = sX[k * kThreads + t] * inv_sumx;
        sX[k * kThreads + t] = X;
        float cf[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) cf[m] = __ldg(md.visc + k * 5 + m);
        const float g = poly4(cf, u);
        const float rg = rcp_approx(g);
        sG[k * kThreads + t] = g;
        sB[k * kThreads + t] = 2.f * X * rg;
        sC[k * kThreads + t] = X * rg * rg;
#pragma unroll
        for (int m = 0; m < 5; ++m) cf[m] = __ldg(md.cond + k * 5 + m);
        const float lk = poly4(cf, u);
        s1 = fmaf(X, lk, s1);
        s2 = fmaf(X, rcp_approx(lk), s2);
    }
    if (lam_o) lam_o[i] = 0.5f * sqrtT * (s1 + rcp_approx(s2));

    if (mu_o) {
        float acc = 0.f;
        for (int k = 0; k < K; ++k) {
            const float gk = sG[k * kThreads + t];
            const float* Bk = md.wilkeB + (size_t)k * K;
            float den = 0.f;
            for (int j = 0; j < K; ++j)
                den = fmaf(__ldg(Bk + j),
                           fmaf(gk, fmaf(gk, sC[j * kThreads + t], sB[j * kThreads + t]), sX[j * kThreads + t]), den);
            acc = fmaf(sX[k * kThreads + t] * __ldg(md.sqrtW + k) * gk * gk, rcp_approx(den), acc);
        }
        mu_o[i] = sqrtT * acc;
    }

    if (D_o) {
        const float p = __ldg(pg + i);
        const float scale = T * sqrtT / p;
        for (int k = 0; k < K; ++k) {
            float S = 0.f, N = 0.f;
            const float* dk = md.dfull + (size_t)k * K * 5;
            for (int j = 0; j < K; ++j) {
                if (j == k) continue;
                float cf[5];
#pragma unroll
                for (int m = 0; m < 5; ++m) cf[m] = __ldg(dk + j * 5 + m);
                S = fmaf(sX[j * kThreads + t], rcp_approx(poly4(cf, u)), S);
                N += __ldg(Yg + (size_t)j * ld + i);
            }
            float Dk;
            if (S > 0.f) {
                Dk = N / S;
            } else {
                float cf[5];
#pragma unroll
                for (int m = 0; m < 5; ++m) cf[m] = __ldg(md.ddiag + k * 5 + m);
                Dk = poly4(cf, u);
            }
            D_o[(size_t)k * ld + i] = Dk * scale;
        }
    }
}

template <int K>
df_status launch_fixed(const PropTables<K>* tab, long long n, long long ld, const float* T, const float* p,
                       const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    const unsigned blocks = (unsigned)((n + kThreads - 1) / kThreads);
    if (mu || lam || D)
        props_fixed_kernel<K, true><<<blocks, kThreads, 0, s>>>(*tab, n, ld, T, p, Y, cp, h, mu, lam, D);
    else
        props_fixed_kernel<K, false><<<blocks, kThreads, 0, s>>>(*tab, n, ld, T, p, Y, cp, h, mu, lam, D);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

}  // namespace

df_status launch_properties(const df_mech* mech, long long n, long long ld, const float* T, const float* p,
                            const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    if ((n + kThreads - 1) / kThreads > 0x7fffffffLL)
        return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_properties: n_cells too large");
    if (mech->t9) return launch_fixed<9>(mech->t9, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    if (mech->t19) return launch_fixed<19>(mech->t19, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    const size_t smem = (size_t)4 * mech->K * kThreads * sizeof(float);
    static bool attr_set = false;
    if (!attr_set) {
        DF_CUDA_TRY(cudaFuncSetAttribute(props_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_set = true;
    }
    const unsigned blocks = (unsigned)((n + kThreads - 1) / kThreads);
    props_generic_kernel<<<blocks, kThreads, smem, s>>>(mech->dev, n, ld, T, p, Y, cp, h, mu, lam, D);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

// properties.cu -- K2: fused mixture thermo + transport pass (NS (2)).
//
// FP32-FMA-bound for every K (12.5 K^2 + 51.5 K flops per cell against 4(2K+6) bytes), so the
// design goal is FMA density, not bytes:
//   * fixed-K kernels (K = 9, 19) take the whole species table as a __grid_constant__ parameter: fully
//     unrolled, coefficients reach the FMAs through uniform registers (LDCU), all per-cell vectors in registers;
//   * Wilke: Phi_kj = B_kj (1 + g_k/g_j)^2 with g = sqrt(mu)/(T W)^(1/4) and B_kj = [8 (1 + W_k/W_j)]^(-1/2) tabulated -- as a
//     truncated singular-value factorisation when the mechanism's weights allow it (R terms: 6 R K instead of 3 K^2 FMAs);
//   * binary diffusion uses each symmetric pair once (4 FFMA Horner + 1 MUFU.RCP + 2 FFMA);
//   * the formation-enthalpy part of h is accumulated in fp64 (K DFMA), the sensible part in fp32.
// Other K (e.g. 53) go to the any-K kernel in properties_group.cu.
#include "common.cuh"

namespace {

constexpr int kThreads = 128;

// ------------------------------------------------------------------------------------------------
// fixed K: two cells per thread, packed fp32x2 arithmetic
// ------------------------------------------------------------------------------------------------
// sm_100a has no constant-bank operand form for FFMA: every table coefficient costs a share of an LDCU/LDC issue
// slot.  Two adjacent cells per thread, held as float2 and updated with FFMA2 (fma.rn.f32x2, whose third form
// broadcasts one scalar uniform register to both halves), halve both the FMA issue slots and the coefficient loads
// per cell.
typedef float2 f2;
__device__ __forceinline__ f2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 fma2(f2 a, float s, f2 c) { return __ffma2_rn(a, bc(s), c); }
__device__ __forceinline__ f2 fma2(float s, f2 a, f2 c) { return __ffma2_rn(bc(s), a, c); }
__device__ __forceinline__ f2 fma2(f2 a, float s, float c) { return __ffma2_rn(a, bc(s), bc(c)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 mul2(f2 a, float s) { return __fmul2_rn(a, bc(s)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
// one MUFU.RCP per half (the shared-reciprocal form 1/x = y/(xy) measured 4 % slower here: its three extra
// multiplies cannot be packed)
__device__ __forceinline__ f2 rcp2(f2 a) { return make_float2(rcp_approx(a.x), rcp_approx(a.y)); }
__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ f2 poly4_2(const float* c, f2 u) {
    return fma2(fma2(fma2(fma2(u, c[4], c[3]), u, bc(c[2])), u, bc(c[1])), u, bc(c[0]));
}

// 4 blocks of 128 threads per SM (128 registers): measured best -- 5 blocks (96 registers) spill 600 B per thread and run
// 19 % slower, 3 blocks (168 registers) 23 % slower
// FULL: every thread of the launch has both of its cells inside the field (the host launches the ragged last block
// separately), so loads and stores are plain float2 accesses without the two-path predicates.
// R: number of terms of Wilke's B in factored form (PropTables::WU, WV), 0 = the full table.
template <int K, bool TRANSPORT, bool FULL, int R>
__global__ void __launch_bounds__(kThreads, 4)
props_fixed_kernel(const __grid_constant__ PropTables<K> tab, long long i_first, long long n, long long ld,
                   const float* __restrict__ Tg, const float* __restrict__ pg, const float* __restrict__ Yg,
                   float* __restrict__ cp_o, float* __restrict__ h_o, float* __restrict__ mu_o,
                   float* __restrict__ lam_o, float* __restrict__ D_o) {
    const long long i = i_first + ((long long)blockIdx.x * kThreads + threadIdx.x) * 2;
    if (!FULL && i >= n) return;
    const bool two = FULL || (i + 1 < n);   // ld % 4 == 0 and 16-byte aligned bases make the float2 accesses legal
    auto ld2 = [&](const float* p) -> f2 {
        if (two) return __ldg(reinterpret_cast<const float2*>(p + i));
        const float v = __ldg(p + i);
        return make_float2(v, v);
    };
    auto st2 = [&](float* p, f2 v) {
        if (two) *reinterpret_cast<float2*>(p + i) = v;
        else p[i] = v.x;
    };
    const f2 T = ld2(Tg);
    f2 Y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) Y[k] = ld2(Yg + (size_t)k * ld);

    // ---- thermo: mixture polynomial in tau, both ranges, select at the end ---------------------
    const f2 tau = mul2(add2(T, bc(-tab.sc.T_mid)), tab.sc.inv_S);
    const bool lo0 = T.x < tab.sc.T_mid, lo1 = T.y < tab.sc.T_mid;  // A2: hi for T >= T_mid
    if (cp_o || h_o) {
        f2 Cl[5], Ch[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) Cl[m] = Ch[m] = bc(0.f);
        double H0l0 = 0.0, H0h0 = 0.0, H0l1 = 0.0, H0h1 = 0.0;
#pragma unroll
        for (int k = 0; k < K; ++k) {
#pragma unroll
            for (int m = 0; m < 5; ++m) {
                Cl[m] = fma2(Y[k], tab.th[k][0][m], Cl[m]);
                Ch[m] = fma2(Y[k], tab.th[k][1][m], Ch[m]);
            }
            H0l0 = fma((double)Y[k].x, tab.h0[k][0], H0l0);
            H0h0 = fma((double)Y[k].x, tab.h0[k][1], H0h0);
            H0l1 = fma((double)Y[k].y, tab.h0[k][0], H0l1);
            H0h1 = fma((double)Y[k].y, tab.h0[k][1], H0h1);
        }
        f2 q[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = make_float2(lo0 ? Cl[m].x : Ch[m].x, lo1 ? Cl[m].y : Ch[m].y);
        const f2 sens = mul2(tau, fma2(fma2(fma2(fma2(q[4], tau, q[3]), tau, q[2]), tau, q[1]), tau, q[0]));
        if (h_o)
            st2(h_o, make_float2((float)((lo0 ? H0l0 : H0h0) + (double)sens.x), (float)((lo1 ? H0l1 : H0h1) + (double)sens.y)));
        if (cp_o)
            st2(cp_o, mul2(fma2(fma2(fma2(fma2(mul2(q[4], 5.f), tau, mul2(q[3], 4.f)), tau, mul2(q[2], 3.f)), tau,
                                     mul2(q[1], 2.f)), tau, q[0]),
                           tab.sc.inv_S));
    }
    if (!TRANSPORT) return;

    // ---- mole fractions -----------------------------------------------------------------------
    f2 X[K];
    f2 sumx = bc(0.f);
#pragma unroll
    for (int k = 0; k < K; ++k) {
        X[k] = mul2(Y[k], tab.invW[k]);
        sumx = add2(sumx, X[k]);
    }
    const f2 inv_sumx = make_float2(1.0f / sumx.x, 1.0f / sumx.y);
#pragma unroll
    for (int k = 0; k < K; ++k) X[k] = mul2(X[k], inv_sumx);

    const f2 u = mul2(add2(make_float2(logf(T.x), logf(T.y)), bc(-tab.sc.Lc)), tab.sc.inv_Ls);
    const f2 sqrtT = make_float2(sqrtf(T.x), sqrtf(T.y));

    // ---- Wilke viscosity ----------------------------------------------------------------------
    if (mu_o && R > 0) {
        // B = sum_m WU[.][m] WV[.][m] (R terms, 1e-6: B is a smooth function of W_k/W_j, its singular values fall ~10x per
        // term): den_k = sum_j B_kj (x_j + 2 g_k x_j r_j + g_k^2 x_j r_j^2), r = 1/g, is evaluated as three projections on the
        // WV_m (3 R K packed FMAs) and K rows from the WU_m (3 R K) instead of 3 K^2; no square roots, X stays X.
        constexpr int RR = R > 0 ? R : 1;
        f2 tP[RR], tQ[RR], tR[RR];
#pragma unroll
        for (int m = 0; m < RR; ++m) tP[m] = tQ[m] = tR[m] = bc(0.f);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const f2 rk = rcp2(poly4_2(tab.visc[k], u));
            const f2 xr = mul2(X[k], rk), xrr = mul2(xr, rk);
#pragma unroll
            for (int m = 0; m < RR; ++m) {
                tP[m] = fma2(X[k], tab.WV[k][m], tP[m]);
                tQ[m] = fma2(xr, tab.WV[k][m], tQ[m]);
                tR[m] = fma2(xrr, tab.WV[k][m], tR[m]);
            }
        }
#pragma unroll
        for (int m = 0; m < RR; ++m) tQ[m] = add2(tQ[m], tQ[m]);
        f2 acc = bc(0.f);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const f2 gk = poly4_2(tab.visc[k], u);
            f2 den = bc(0.f);
#pragma unroll
            for (int m = 0; m < RR; ++m) den = fma2(fma2(gk, fma2(gk, tR[m], tQ[m]), tP[m]), tab.WU[k][m], den);
            acc = fma2(mul2(mul2(X[k], tab.sqrtW[k]), mul2(gk, gk)), rcp2(den), acc);
        }
        st2(mu_o, mul2(sqrtT, acc));
    }
    if (mu_o && R == 0) {
        // x_j Phi_kj = B_kj (sqrt(x_j) + g_k sqrt(x_j)/g_j)^2: two per-species vectors (a_j = sqrt(x_j), b_j = a_j/g_j) and
        // 3 packed instructions per (k,j) -- the register footprint of the two-vector form at the instruction count of the
        // three-vector one.  X_j is rebuilt as a_j^2 afterwards (1 ulp; exact for x_j = 0).
        f2 b[K];
        f2 acc = bc(0.f);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            X[k] = make_float2(sqrt_approx(X[k].x), sqrt_approx(X[k].y));
            b[k] = mul2(X[k], rcp2(poly4_2(tab.visc[k], u)));
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const f2 gk = poly4_2(tab.visc[k], u);
            f2 den = bc(0.f);
#pragma unroll
            for (int j = 0; j < K; ++j) {
                const f2 t = fma2(gk, b[j], X[j]);
                den = fma2(mul2(t, t), tab.B[k][j], den);
            }
            acc = fma2(mul2(mul2(mul2(X[k], X[k]), tab.sqrtW[k]), mul2(gk, gk)), rcp2(den), acc);
        }
#pragma unroll
        for (int k = 0; k < K; ++k) X[k] = mul2(X[k], X[k]);
        st2(mu_o, mul2(sqrtT, acc));
    }

    // ---- combination-rule conductivity (A6) ---------------------------------------------------
    if (lam_o) {
        f2 s1 = bc(0.f), s2 = bc(0.f);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const f2 lk = poly4_2(tab.cond[k], u);
            s1 = fma2(X[k], lk, s1);
            s2 = fma2(X[k], rcp2(lk), s2);
        }
        st2(lam_o, mul2(mul2(sqrtT, 0.5f), add2(s1, rcp2(s2))));
    }

    // ---- mixture-averaged diffusivities (A7) ---------------------------------------------
    if (D_o) {
        const f2 p = ld2(pg);
        const f2 scale = mul2(mul2(T, sqrtT), rcp2(p));
        f2 S[K];
#pragma unroll
        for (int k = 0; k < K; ++k) S[k] = bc(0.f);
        {
            // one MUFU per half and pair; sharing a reciprocal between two pairs (1/a = b/(ab): 2 MUFU + 3 packed multiplies
            // for 4 MUFU) on any share of the pairs measured no faster (0.273-0.277 ms): the loop waits on latency, not on the XU
            int idx = 0;
#pragma unroll
            for (int j = 0; j < K; ++j)
#pragma unroll
                for (int k = j + 1; k < K; ++k, ++idx) {
                    const f2 r = rcp2(poly4_2(tab.dpair[idx], u));
                    S[k] = fma2(X[j], r, S[k]);
                    S[j] = fma2(X[k], r, S[j]);
                }
        }
        // N_k = sum_{j != k} Y_j as prefix + suffix (never 1 - Y_k: cancels when Y_k -> 1).  Y is re-read here (L2 hit)
        // instead of being kept live through the Wilke block: 38 registers less at the kernel's pressure peak.
#pragma unroll
        for (int k = 0; k < K; ++k) Y[k] = ld2(Yg + (size_t)k * ld);
        f2 suf[K + 1];
        suf[K] = bc(0.f);
#pragma unroll
        for (int k = K - 1; k >= 0; --k) suf[k] = add2(suf[k + 1], Y[k]);
        f2 pre = bc(0.f);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const f2 Nk = add2(pre, suf[k + 1]);
            pre = add2(pre, Y[k]);
            const f2 dk = poly4_2(tab.ddiag[k], u);
            // MUFU reciprocal (1e-7) instead of the IEEE division: the 2 x 19 divisions were 17 % of the kernel's PC samples
            const f2 q = mul2(Nk, rcp2(S[k]));
            const f2 Dk = make_float2(S[k].x > 0.f ? q.x : dk.x, S[k].y > 0.f ? q.y : dk.y);
            st2(D_o + (size_t)k * ld, mul2(Dk, scale));
        }
    }
}

template <int K, int R>
df_status launch_fixed_r(const PropTables<K>* tab, long long n, long long ld, const float* T, const float* p,
                         const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    constexpr long long per_block = 2 * kThreads;
    const long long full_blocks = n / per_block, tail_first = full_blocks * per_block;
    const bool transport = mu || lam || D;
    if (full_blocks > 0) {
        if (transport) props_fixed_kernel<K, true, true, R><<<(unsigned)full_blocks, kThreads, 0, s>>>(*tab, 0, n, ld, T, p, Y, cp, h, mu, lam, D);
        else props_fixed_kernel<K, false, true, 0><<<(unsigned)full_blocks, kThreads, 0, s>>>(*tab, 0, n, ld, T, p, Y, cp, h, mu, lam, D);
    }
    if (tail_first < n) {   // the ragged last block
        if (transport) props_fixed_kernel<K, true, false, R><<<1, kThreads, 0, s>>>(*tab, tail_first, n, ld, T, p, Y, cp, h, mu, lam, D);
        else props_fixed_kernel<K, false, false, 0><<<1, kThreads, 0, s>>>(*tab, tail_first, n, ld, T, p, Y, cp, h, mu, lam, D);
    }
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

template <int K>
df_status launch_fixed(const PropTables<K>* tab, long long n, long long ld, const float* T, const float* p,
                       const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    if constexpr (K > 16) {   // the factored Wilke when the mechanism's B allows it (mech.cu: make_fixed)
        if (tab->wilke_rank == 7) return launch_fixed_r<K, 7>(tab, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        if (tab->wilke_rank == 8) return launch_fixed_r<K, 8>(tab, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    }
    return launch_fixed_r<K, 0>(tab, n, ld, T, p, Y, cp, h, mu, lam, D, s);
}

}  // namespace

df_status launch_properties(const df_mech* mech, long long n, long long ld, const float* T, const float* p,
                            const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    if ((n + kThreads - 1) / kThreads > 0x7fffffffLL)
        return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_properties: n_cells too large");
    if (mech->t9) return launch_fixed<9>(mech->t9, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    if (mech->t19) return launch_fixed<19>(mech->t19, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    return launch_properties_group(mech, n, ld, T, p, Y, cp, h, mu, lam, D, s);
}

// properties_tiled.cu -- K2 for any species count K <= 64 (BASELINE config 4: K = 53).
//
// At K = 53 the per-cell vectors (X, 1/g, S: 3 x 53 values) no longer fit in registers, and a fully unrolled
// kernel would be ~20 k instructions, so this kernel tiles the O(K^2) work:
//   * one thread owns two adjacent cells as float2 (packed FFMA2 arithmetic, see properties.cu);
//   * the per-cell vectors live in shared memory as [species][thread] (conflict-free), species padded to a
//     multiple of 8 with inert entries (X = 0) so the tile loops have no remainder code;
//   * Wilke: 8 accumulators den_k per k-tile in registers, j streams from shared memory, B_kj arrives as two
//     warp-uniform float4 loads per j (the table is stored transposed for that);
//   * binary diffusion: 8 x 8 register tiles over the upper triangle of (k, j); each pair is evaluated once
//     (4 FFMA2 Horner, one MUFU.RCP for both cells, 2 FFMA2) and scattered to S_k (registers) and S_j (registers,
//     flushed to shared memory once per tile); the 8 coefficients of a pair are two warp-uniform float4 loads from
//     a table pre-tiled in exactly this order;
//   * N_k = sum_{j != k} Y_j = prefix + suffix (suffix sums parked in the output array): no 1 - Y_k cancellation (A7).
#include "common.cuh"

namespace {

constexpr int kTT = 64;  // threads per block (2 cells each)
typedef float2 f2;
__device__ __forceinline__ f2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 fma2(f2 a, float s, f2 c) { return __ffma2_rn(a, bc(s), c); }
__device__ __forceinline__ f2 fma2(f2 a, float s, float c) { return __ffma2_rn(a, bc(s), bc(c)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 mul2(f2 a, float s) { return __fmul2_rn(a, bc(s)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
// reciprocals of both halves from one MUFU: 1/x = y/(xy), 1/y = x/(xy)
__device__ __forceinline__ f2 rcp2(f2 a) {
    const float r = rcp_approx(a.x * a.y);
    return make_float2(r * a.y, r * a.x);
}
__device__ __forceinline__ f2 poly4_2(float c0, float c1, float c2, float c3, float c4, f2 u) {
    return fma2(fma2(fma2(fma2(u, c4, c3), u, bc(c2)), u, bc(c1)), u, bc(c0));
}

template <bool DIAG>
__device__ __forceinline__ void diff_tile(const float* __restrict__ coef, f2 u, const f2 (&Xk)[8], const f2 (&Xj)[8],
                                          f2 (&Sk)[8], f2 (&Sj)[8]) {
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = DIAG ? a + 1 : 0; b < 8; ++b) {
            const float4 c0 = *reinterpret_cast<const float4*>(coef + (a * 8 + b) * 8);   // warp-uniform: broadcast LDS
            const float c4 = coef[(a * 8 + b) * 8 + 4];
            const f2 r = rcp2(poly4_2(c0.x, c0.y, c0.z, c0.w, c4, u));
            Sk[a] = fma2(Xj[b], r, Sk[a]);
            Sj[b] = fma2(Xk[a], r, Sj[b]);
        }
}

__global__ void __launch_bounds__(kTT)
props_tiled_kernel(MechDev md, long long n, long long ld, const float* __restrict__ Tg, const float* __restrict__ pg,
                   const float* __restrict__ Yg, float* __restrict__ cp_o, float* __restrict__ h_o,
                   float* __restrict__ mu_o, float* __restrict__ lam_o, float* __restrict__ D_o) {
    extern __shared__ float2 sm2[];
    const int K = md.K, Kp = md.Kp, nt = Kp >> 3, t = threadIdx.x;
    f2* sX = sm2;                 // [Kp][kTT] mole fractions
    f2* sR = sX + Kp * kTT;       // 1/g (Wilke), then the S_k accumulators (diffusion)
    float* sBT = reinterpret_cast<float*>(sR + Kp * kTT);   // [Kp][Kp] Wilke table (transposed), staged once per block
    float* sCo = sBT + Kp * Kp;                             // [2][512] double-buffered diffusion coefficient tiles
    // every thread stays alive (the tile staging below uses block-wide barriers); threads past the end of the field
    // work on cell 0 and do not store
    const long long i_raw = ((long long)blockIdx.x * kTT + t) * 2;
    const bool valid = i_raw < n;
    const long long i = valid ? i_raw : 0;
    const bool two = valid && (i + 1 < n);
    for (int e = t; e < Kp * Kp / 4; e += kTT)
        reinterpret_cast<float4*>(sBT)[e] = __ldg(reinterpret_cast<const float4*>(md.BT) + e);
    auto ld2 = [&](const float* p) -> f2 {
        if (two) return __ldg(reinterpret_cast<const float2*>(p + i));
        const float v = __ldg(p + i);
        return make_float2(v, v);
    };
    auto st2 = [&](float* p, f2 v) {
        if (two) *reinterpret_cast<float2*>(p + i) = v;
        else if (valid) p[i] = v.x;
    };
    const f2 T = ld2(Tg);
    const f2 tau = mul2(add2(T, bc(-md.sc.T_mid)), md.sc.inv_S);
    const bool lo0 = T.x < md.sc.T_mid, lo1 = T.y < md.sc.T_mid;

    // ---- phase 1: thermo (both ranges, select at the end), x_k = Y_k / W_k -----------------------------------
    f2 Cl[5], Ch[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) Cl[m] = Ch[m] = bc(0.f);
    double H0l0 = 0.0, H0h0 = 0.0, H0l1 = 0.0, H0h1 = 0.0;
    f2 sumx = bc(0.f);
#pragma unroll 8
    for (int k = 0; k < K; ++k) {   // unrolled: eight rounds of (L2-latency) loads in flight per thread
        const f2 y = ld2(Yg + (size_t)k * ld);
        const float4* th = reinterpret_cast<const float4*>(md.thp + k * 12);
        const float4 a = __ldg(th), b = __ldg(th + 1), c = __ldg(th + 2);  // lo c0..c5 | hi c0..c5
        Cl[0] = fma2(y, a.y, Cl[0]); Cl[1] = fma2(y, a.z, Cl[1]); Cl[2] = fma2(y, a.w, Cl[2]);
        Cl[3] = fma2(y, b.x, Cl[3]); Cl[4] = fma2(y, b.y, Cl[4]);
        Ch[0] = fma2(y, b.w, Ch[0]); Ch[1] = fma2(y, c.x, Ch[1]); Ch[2] = fma2(y, c.y, Ch[2]);
        Ch[3] = fma2(y, c.z, Ch[3]); Ch[4] = fma2(y, c.w, Ch[4]);
        if (h_o) {
            const double hl = __ldg(md.h0p + 2 * k), hh = __ldg(md.h0p + 2 * k + 1);
            H0l0 = fma((double)y.x, hl, H0l0); H0h0 = fma((double)y.x, hh, H0h0);
            H0l1 = fma((double)y.y, hl, H0l1); H0h1 = fma((double)y.y, hh, H0h1);
        }
        const f2 x = mul2(y, __ldg(md.small_p + k * 24));
        sX[k * kTT + t] = x;
        sumx = add2(sumx, x);
    }
    for (int k = K; k < Kp; ++k) sX[k * kTT + t] = bc(0.f);
    if (cp_o || h_o) {
        f2 q[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) q[m] = make_float2(lo0 ? Cl[m].x : Ch[m].x, lo1 ? Cl[m].y : Ch[m].y);
        const f2 sens = mul2(tau, fma2(fma2(fma2(fma2(q[4], tau, q[3]), tau, q[2]), tau, q[1]), tau, q[0]));
        if (h_o)
            st2(h_o, make_float2((float)((lo0 ? H0l0 : H0h0) + (double)sens.x), (float)((lo1 ? H0l1 : H0h1) + (double)sens.y)));
        if (cp_o)
            st2(cp_o, mul2(fma2(fma2(fma2(fma2(mul2(q[4], 5.f), tau, mul2(q[3], 4.f)), tau, mul2(q[2], 3.f)), tau,
                                     mul2(q[1], 2.f)), tau, q[0]),
                           md.sc.inv_S));
    }
    if (!mu_o && !lam_o && !D_o) return;   // block-uniform
    __syncthreads();                       // sBT is staged

    // ---- phase 2: X_k, r_k = 1/g_k, conductivity ---------------------------------------------------------------
    const f2 inv_sumx = make_float2(1.0f / sumx.x, 1.0f / sumx.y);
    const f2 u = mul2(add2(make_float2(logf(T.x), logf(T.y)), bc(-md.sc.Lc)), md.sc.inv_Ls);
    const f2 sqrtT = make_float2(sqrtf(T.x), sqrtf(T.y));
    {
        f2 s1 = bc(0.f), s2 = bc(0.f);
#pragma unroll 8
        for (int k = 0; k < Kp; ++k) {
            const f2 X = mul2(sX[k * kTT + t], inv_sumx);
            sX[k * kTT + t] = X;
            const float4* sp = reinterpret_cast<const float4*>(md.small_p + k * 24);
            const float4 a = __ldg(sp), b = __ldg(sp + 1), c = __ldg(sp + 2);  // invW sqrtW v0 v1 | v2 v3 v4 c0 | c1 c2 c3 c4
            sR[k * kTT + t] = rcp2(poly4_2(a.z, a.w, b.x, b.y, b.z, u));
            const f2 lk = poly4_2(b.w, c.x, c.y, c.z, c.w, u);
            s1 = fma2(X, lk, s1);
            s2 = fma2(X, rcp2(lk), s2);
        }
        if (lam_o) st2(lam_o, mul2(mul2(sqrtT, 0.5f), add2(s1, rcp2(s2))));
    }

    // ---- phase 3: Wilke, Phi_kj = B_kj (1 + g_k r_j)^2 ----------------------------------------------------------
    if (mu_o) {
        f2 acc = bc(0.f);
        for (int kt = 0; kt < nt; ++kt) {
            const int k0 = kt * 8;
            f2 gk[8], den[8];
#pragma unroll
            for (int a = 0; a < 8; ++a) {
                gk[a] = rcp2(sR[(k0 + a) * kTT + t]);
                den[a] = bc(0.f);
            }
#pragma unroll 2
            for (int j = 0; j < Kp; ++j) {
                const f2 xj = sX[j * kTT + t], rj = sR[j * kTT + t];
                const float4* bt = reinterpret_cast<const float4*>(sBT + j * Kp + k0);
                const float4 b0 = bt[0], b1 = bt[1];
                const float B[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
                for (int a = 0; a < 8; ++a) {
                    const f2 tt = fma2(gk[a], rj, bc(1.0f));
                    den[a] = fma2(mul2(xj, mul2(tt, tt)), B[a], den[a]);
                }
            }
#pragma unroll
            for (int a = 0; a < 8; ++a) {
                const float sw = __ldg(md.small_p + (k0 + a) * 24 + 1);
                acc = fma2(mul2(mul2(sX[(k0 + a) * kTT + t], sw), mul2(gk[a], gk[a])), rcp2(den[a]), acc);
            }
        }
        st2(mu_o, mul2(sqrtT, acc));
    }

    // ---- phase 4: mixture-averaged diffusivities ---------------------------------------------------------------
    if (D_o) {
        const f2 p = ld2(pg);
        const f2 scale = make_float2(T.x * sqrtT.x / p.x, T.y * sqrtT.y / p.y);
        {
            f2 suf = bc(0.f);
            // suffix sums sum_{j > k} Y_j are parked in the output array (read back, then overwritten, below):
            // a third per-thread vector in shared memory would cost a third of the occupancy
#pragma unroll 8
            for (int k = Kp - 1; k >= 0; --k) {
                sR[k * kTT + t] = bc(0.f);
                if (k < K) {
                    st2(D_o + (size_t)k * ld, suf);
                    suf = add2(suf, ld2(Yg + (size_t)k * ld));
                }
            }
        }
        f2 pre = bc(0.f);
        // coefficient tiles (2 KB each, in loop order) are staged through shared memory, double-buffered: the whole
        // block copies tile tix + 1 while it computes tile tix
        const float4* gco = reinterpret_cast<const float4*>(md.dtile);
        const int ntiles = nt * (nt + 1) / 2;
        reinterpret_cast<float4*>(sCo)[t] = __ldg(gco + t);
        reinterpret_cast<float4*>(sCo)[t + kTT] = __ldg(gco + t + kTT);
        __syncthreads();
        int tix = 0;
        for (int kt = 0; kt < nt; ++kt) {
            const int k0 = kt * 8;
            f2 Xk[8], Sk[8];
#pragma unroll
            for (int a = 0; a < 8; ++a) {
                Xk[a] = sX[(k0 + a) * kTT + t];
                Sk[a] = bc(0.f);
            }
            for (int jt = kt; jt < nt; ++jt, ++tix) {
                const int j0 = jt * 8;
                const float* coef = sCo + (tix & 1) * 512;
                float4 n0, n1;
                const bool more = tix + 1 < ntiles;
                if (more) {
                    n0 = __ldg(gco + (size_t)(tix + 1) * 128 + t);
                    n1 = __ldg(gco + (size_t)(tix + 1) * 128 + t + kTT);
                }
                f2 Xj[8], Sj[8];
#pragma unroll
                for (int b = 0; b < 8; ++b) {
                    Xj[b] = sX[(j0 + b) * kTT + t];
                    Sj[b] = bc(0.f);
                }
                if (jt == kt) diff_tile<true>(coef, u, Xk, Xj, Sk, Sj);
                else diff_tile<false>(coef, u, Xk, Xj, Sk, Sj);
#pragma unroll
                for (int b = 0; b < 8; ++b) sR[(j0 + b) * kTT + t] = add2(sR[(j0 + b) * kTT + t], Sj[b]);
                if (more) {
                    float4* dst = reinterpret_cast<float4*>(sCo + ((tix + 1) & 1) * 512);
                    dst[t] = n0;
                    dst[t + kTT] = n1;
                }
                __syncthreads();
            }
#pragma unroll
            for (int a = 0; a < 8; ++a) {
                const int k = k0 + a;
                if (k < K) {
                    const f2 S = add2(Sk[a], sR[k * kTT + t]);
                    const f2 Nk = add2(pre, two ? *reinterpret_cast<const float2*>(D_o + (size_t)k * ld + i)
                                                : bc(D_o[(size_t)k * ld + i]));
                    pre = add2(pre, ld2(Yg + (size_t)k * ld));
                    const float* dd = md.small_p + k * 24 + 12;
                    const f2 dk = poly4_2(__ldg(dd), __ldg(dd + 1), __ldg(dd + 2), __ldg(dd + 3), __ldg(dd + 4), u);
                    const f2 Dk = make_float2(S.x > 0.f ? Nk.x / S.x : dk.x, S.y > 0.f ? Nk.y / S.y : dk.y);
                    st2(D_o + (size_t)k * ld, mul2(Dk, scale));
                }
            }
        }
    }
}

}  // namespace

df_status launch_properties_tiled(const df_mech* mech, long long n, long long ld, const float* T, const float* p,
                                  const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    const MechDev& md = mech->dev;
    const size_t smem = (size_t)2 * md.Kp * kTT * sizeof(float2) + ((size_t)md.Kp * md.Kp + 1024) * sizeof(float);
    static DfPerDevice smem_attr;
    const df_status st = df_ensure_dyn_smem((const void*)props_tiled_kernel, 200 * 1024, &smem_attr);
    if (st != DF_OK) return st;
    const long long blocks = (n + 2 * kTT - 1) / (2 * kTT);
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_properties: n_cells too large");
    props_tiled_kernel<<<(unsigned)blocks, kTT, smem, s>>>(md, n, ld, T, p, Y, cp, h, mu, lam, D);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

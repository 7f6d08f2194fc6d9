// pointwise.cu -- the two HBM-bound per-cell passes around the property and ANN calls:
//   df_thermo_extras      rho, psi = Wbar/(R T), alpha = lambda/cp, rho D_k, h_k(T), mixture entropy   (reading A22)
//   df_chem_pasr_scale    PaSR factor kappa = tau_c/(tau_c + tau_mix) applied to omega_k, with the T gate (A23)
// One thread owns four consecutive cells (float4 SoA accesses, 512 B per warp and species row); the species tables
// (<= 7 KB) are staged in shared memory once per block; every input row is read once (single pass: rho factors out of
// the PaSR time scale, the entropy of mixing is split as sum x ln x - (1/Wbar) ln(1/Wbar)), so the DRAM traffic is the
// algorithmic 4 B per field element.
#include "common.cuh"

namespace {

constexpr int kPT = 128;   // threads per block, 4 cells each

struct F4 {
    float v[4];
};
// FULL (template parameter of the kernels): all four cells of every thread are inside the field -- the ragged last
// block is launched separately -- so the accesses are plain float4 without the two-path branch.
template <bool FULL>
__device__ __forceinline__ F4 load4(const float* __restrict__ p, long long i0, long long n, float fill) {
    F4 r;
    if (FULL || i0 + 4 <= n) {
        const float4 t = __ldg(reinterpret_cast<const float4*>(p + i0));
        r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c) r.v[c] = (i0 + c < n) ? __ldg(p + i0 + c) : fill;
    }
    return r;
}
template <bool FULL>
__device__ __forceinline__ void store4(float* __restrict__ p, long long i0, long long n, const F4& r) {
    if (FULL || i0 + 4 <= n) {
        *reinterpret_cast<float4*>(p + i0) = make_float4(r.v[0], r.v[1], r.v[2], r.v[3]);
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (i0 + c < n) p[i0 + c] = r.v[c];
    }
}

// species rows (float4 per thread) loaded ahead of their use in every pass: the passes are HBM-bound and a row-at-a-time
// loop leaves too few bytes in flight (extras 0.165 -> 0.135 ms, pasr -7 %; 2 and 8 rows measured slower)
constexpr int kRowsAhead = 4;
// ---- NEXT-4 ------------------------------------------------------------------------------------------------------
template <bool FULL>
__global__ void __launch_bounds__(kPT)
extras_kernel(MechDev md, long long i_first, long long n, long long ld, const float* __restrict__ Tg, const float* __restrict__ pg,
              const float* __restrict__ Yg, const float* __restrict__ cpg, const float* __restrict__ lamg,
              const float* __restrict__ Dg, float* __restrict__ rho_o, float* __restrict__ psi_o,
              float* __restrict__ alpha_o, float* __restrict__ rhoD_o, float* __restrict__ hk_o, float* __restrict__ s_o) {
    extern __shared__ float sm[];
    const int K = md.K;
    float* sTh = sm;                 // [K][2][6]  h_k/W_k in tau
    float* sS = sTh + K * 12;        // [K][2][6]  s_k/W_k: coefficient of ln T, then the polynomial part in tau
    float* sIW = sS + K * 12;        // [K] 1/W_k
    for (int e = threadIdx.x; e < K * 12; e += kPT) {
        sTh[e] = md.th32[e];
        sS[e] = md.sth32[e];
    }
    for (int e = threadIdx.x; e < K; e += kPT) sIW[e] = md.invW[e];
    __syncthreads();
    const long long i0 = i_first + ((long long)blockIdx.x * kPT + threadIdx.x) * 4;
    if (!FULL && i0 >= n) return;
    const F4 T = load4<FULL>(Tg, i0, n, 1000.f), p = load4<FULL>(pg, i0, n, 101325.f);

    // ONE pass over Y: 1/Wbar and, when the entropy is wanted, sum_k Y_k s_k(T) and sum_k x_k ln x_k (x_k = Y_k/W_k):
    //   s = sum_k Y_k s_k/W_k - R sum_k x_k ln(x_k Wbar) - (R/Wbar) ln(p/p0)
    //     = sum_k Y_k s_k/W_k - R [sum_k x_k ln x_k - (1/Wbar) ln(1/Wbar)] - (R/Wbar) ln(p/p0)
    float lnT[4], tau[4];
    int lo[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        lnT[c] = logf(T.v[c]);
        tau[c] = (T.v[c] - md.sc.T_mid) * md.sc.inv_S;
        lo[c] = T.v[c] < md.sc.T_mid;   // A2
    }
    float invWbar[4] = {0.f, 0.f, 0.f, 0.f}, sy[4] = {0.f, 0.f, 0.f, 0.f}, sxlx[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k0 = 0; k0 < K; k0 += kRowsAhead) {   // kRowsAhead rows of Y in flight at once
        F4 yq[kRowsAhead];
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q)
            if (k0 + q < K) yq[q] = load4<FULL>(Yg + (size_t)(k0 + q) * ld, i0, n, 0.f);
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q) {
            const int k = k0 + q;
            if (k >= K) break;
            const F4 y = yq[q];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float x = y.v[c] * sIW[k];
                invWbar[c] += x;
                if (s_o) {
                    const float* q6 = sS + k * 12 + (lo[c] ? 0 : 6);
                    const float sk = fmaf(q6[0], lnT[c], fmaf(fmaf(fmaf(fmaf(q6[5], tau[c], q6[4]), tau[c], q6[3]), tau[c], q6[2]), tau[c], q6[1]));
                    sy[c] = fmaf(y.v[c], sk, sy[c]);
                    sxlx[c] += x > 0.f ? x * __logf(x) : 0.f;   // x ln x -> 0; MUFU lg2: |err| < 1e-6 on a term that is ~1 % of s
                }
            }
        }
    }
    const float Ru = (float)DF_R_UNIVERSAL;
    F4 rho, psi;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        psi.v[c] = 1.0f / (invWbar[c] * Ru * T.v[c]);
        rho.v[c] = p.v[c] * psi.v[c];
    }
    if (rho_o) store4<FULL>(rho_o, i0, n, rho);
    if (psi_o) store4<FULL>(psi_o, i0, n, psi);
    if (alpha_o) {
        const F4 cp = load4<FULL>(cpg, i0, n, 1.f), lam = load4<FULL>(lamg, i0, n, 0.f);
        F4 a;
#pragma unroll
        for (int c = 0; c < 4; ++c) a.v[c] = lam.v[c] / cp.v[c];
        store4<FULL>(alpha_o, i0, n, a);
    }
    if (s_o) {
        F4 o;
#pragma unroll
        for (int c = 0; c < 4; ++c)
            o.v[c] = sy[c] - Ru * (sxlx[c] - invWbar[c] * logf(invWbar[c])) - Ru * invWbar[c] * logf(p.v[c] * (1.0f / 101325.0f));
        store4<FULL>(s_o, i0, n, o);
    }
    if (!rhoD_o && !hk_o) return;
    // kRowsAhead rows of D in flight at once
    for (int k0 = 0; k0 < K; k0 += kRowsAhead) {
        F4 d[kRowsAhead];
        if (rhoD_o) {
#pragma unroll
            for (int q = 0; q < kRowsAhead; ++q)
                if (k0 + q < K) d[q] = load4<FULL>(Dg + (size_t)(k0 + q) * ld, i0, n, 0.f);
        }
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q) {
            const int k = k0 + q;
            if (k >= K) break;
            if (rhoD_o) {
                F4 o;
#pragma unroll
                for (int c = 0; c < 4; ++c) o.v[c] = rho.v[c] * d[q].v[c];
                store4<FULL>(rhoD_o + (size_t)k * ld, i0, n, o);
            }
            if (hk_o) {
                F4 o;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float* q6 = sTh + k * 12 + (lo[c] ? 0 : 6);
                    o.v[c] = fmaf(fmaf(fmaf(fmaf(fmaf(q6[5], tau[c], q6[4]), tau[c], q6[3]), tau[c], q6[2]), tau[c], q6[1]), tau[c], q6[0]);
                }
                store4<FULL>(hk_o + (size_t)k * ld, i0, n, o);
            }
        }
    }
}

// ---- NEXT-3 ------------------------------------------------------------------------------------------------------
// One pass over Y and omega: rho factors out of the slowest time scale, tau_c = rho max_k Y_k/|omega_k|; the omega rows
// are read again for the scaling (a variant that kept them in registers for K <= 24 needed 140 registers and ran 45 %
// slower: the occupancy is worth more than the 4 K bytes per cell, which come from L2 mostly).
template <bool FULL>
__global__ void __launch_bounds__(kPT)
pasr_kernel(MechDev md, long long i_first, long long n, long long ld, const float* __restrict__ Tg, const float* __restrict__ pg,
            const float* __restrict__ Yg, const float* __restrict__ mug, const float* __restrict__ kg,
            const float* __restrict__ eg, float T_gate, float* omega, float* __restrict__ kappa_o) {
    extern __shared__ float sm[];
    const int K = md.K;
    for (int e = threadIdx.x; e < K; e += kPT) sm[e] = md.invW[e];
    __syncthreads();
    const long long i0 = i_first + ((long long)blockIdx.x * kPT + threadIdx.x) * 4;
    if (!FULL && i0 >= n) return;
    const F4 T = load4<FULL>(Tg, i0, n, 1000.f), p = load4<FULL>(pg, i0, n, 101325.f);
    float invWbar[4] = {0.f, 0.f, 0.f, 0.f}, m[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k0 = 0; k0 < K; k0 += kRowsAhead) {   // kRowsAhead rows of Y and omega in flight at once
        F4 yq[kRowsAhead], wq[kRowsAhead];
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q)
            if (k0 + q < K) {
                yq[q] = load4<FULL>(Yg + (size_t)(k0 + q) * ld, i0, n, 0.f);
                wq[q] = load4<FULL>(omega + (size_t)(k0 + q) * ld, i0, n, 0.f);
            }
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q) {
            if (k0 + q >= K) break;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                invWbar[c] = fmaf(yq[q].v[c], sm[k0 + q], invWbar[c]);
                const float a = fabsf(wq[q].v[c]);
                if (a > 0.f) m[c] = fmaxf(m[c], yq[q].v[c] * rcp_approx(a));   // species that do not react do not count
            }
        }
    }
    const F4 mu = load4<FULL>(mug, i0, n, 1.f), ks = load4<FULL>(kg, i0, n, 1.f), ep = load4<FULL>(eg, i0, n, 1.f);
    F4 kappa;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float rho = p.v[c] * rcp_approx(invWbar[c] * (float)DF_R_UNIVERSAL * T.v[c]);
        const float tau_c = rho * m[c];
        const float re = rcp_approx(ep.v[c]);
        const float tau_mix = sqrtf(ks.v[c] * re * sqrtf(mu.v[c] * re * rcp_approx(rho)));
        float kp = tau_c > 0.f ? tau_c * rcp_approx(tau_c + tau_mix) : 0.f;
        if (T.v[c] < T_gate) kp = 0.f;
        kappa.v[c] = kp;
    }
    if (kappa_o) store4<FULL>(kappa_o, i0, n, kappa);
    for (int k0 = 0; k0 < K; k0 += kRowsAhead) {
        F4 wq[kRowsAhead];
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q)
            if (k0 + q < K) wq[q] = load4<FULL>(omega + (size_t)(k0 + q) * ld, i0, n, 0.f);
#pragma unroll
        for (int q = 0; q < kRowsAhead; ++q) {
            if (k0 + q >= K) break;
#pragma unroll
            for (int c = 0; c < 4; ++c) wq[q].v[c] *= kappa.v[c];
            store4<FULL>(omega + (size_t)(k0 + q) * ld, i0, n, wq[q]);
        }
    }
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

df_status check(const char* fn, const df_mech* mech, long long n, long long ld) {
    if (!mech) return df_set_error(DF_ERR_INVALID_ARG, "%s: mech is NULL", fn);
    if (n < 0) return df_set_error(DF_ERR_INVALID_ARG, "%s: n_cells < 0", fn);
    if (ld < n) return df_set_error(DF_ERR_INVALID_ARG, "%s: ld (%lld) < n_cells (%lld)", fn, ld, n);
    if (ld % 4 != 0) return df_set_error(DF_ERR_INVALID_ARG, "%s: ld (%lld) must be a multiple of 4", fn, ld);
    if ((n + 4LL * kPT - 1) / (4LL * kPT) > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "%s: n_cells too large", fn);
    return DF_OK;
}

}  // namespace

extern "C" df_status df_thermo_extras(const df_mech* mech, long long n, long long ld, const float* T, const float* p,
                                      const float* Y, const float* cp, const float* lambda, const float* D, float* rho,
                                      float* psi, float* alpha, float* rhoD, float* hk, float* s, void* stream) {
    const df_status st = check("df_thermo_extras", mech, n, ld);
    if (st != DF_OK) return st;
    if (n == 0) return DF_OK;
    if (!T || !p || !Y) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_extras: NULL input field");
    if (alpha && (!cp || !lambda)) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_extras: alpha needs cp and lambda");
    if (rhoD && !D) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_extras: rhoD needs D");
    if (!rho && !psi && !alpha && !rhoD && !hk && !s) return DF_OK;
    const void* ptrs[] = {T, p, Y, cp, lambda, D, rho, psi, alpha, rhoD, hk, s};
    for (const void* q : ptrs)
        if (!aligned16(q)) return df_set_error(DF_ERR_INVALID_ARG, "df_thermo_extras: fields must be 16-byte aligned");
    const long long full_blocks = n / (4LL * kPT), tail_first = full_blocks * 4LL * kPT;
    const size_t smem = (size_t)mech->K * 25 * sizeof(float);
    if (full_blocks > 0)
        extras_kernel<true><<<(unsigned)full_blocks, kPT, smem, (cudaStream_t)stream>>>(mech->dev, 0, n, ld, T, p, Y, cp, lambda, D, rho, psi,
                                                                                       alpha, rhoD, hk, s);
    if (tail_first < n)
        extras_kernel<false><<<1, kPT, smem, (cudaStream_t)stream>>>(mech->dev, tail_first, n, ld, T, p, Y, cp, lambda, D, rho, psi, alpha,
                                                                     rhoD, hk, s);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

extern "C" df_status df_chem_pasr_scale(const df_mech* mech, long long n, long long ld, const float* T, const float* p,
                                        const float* Y, const float* mu, const float* k_sgs, const float* eps, float T_gate,
                                        float* omega, float* kappa, void* stream) {
    const df_status st = check("df_chem_pasr_scale", mech, n, ld);
    if (st != DF_OK) return st;
    if (n == 0) return DF_OK;
    if (!T || !p || !Y || !mu || !k_sgs || !eps || !omega) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_pasr_scale: NULL field");
    const void* ptrs[] = {T, p, Y, mu, k_sgs, eps, omega, kappa};
    for (const void* q : ptrs)
        if (!aligned16(q)) return df_set_error(DF_ERR_INVALID_ARG, "df_chem_pasr_scale: fields must be 16-byte aligned");
    const long long full_blocks = n / (4LL * kPT), tail_first = full_blocks * 4LL * kPT;
    const size_t smem = (size_t)mech->K * sizeof(float);
    if (full_blocks > 0)
        pasr_kernel<true><<<(unsigned)full_blocks, kPT, smem, (cudaStream_t)stream>>>(mech->dev, 0, n, ld, T, p, Y, mu, k_sgs, eps, T_gate,
                                                                                     omega, kappa);
    if (tail_first < n)
        pasr_kernel<false><<<1, kPT, smem, (cudaStream_t)stream>>>(mech->dev, tail_first, n, ld, T, p, Y, mu, k_sgs, eps, T_gate, omega, kappa);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

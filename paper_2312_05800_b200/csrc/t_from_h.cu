// t_from_h.cu -- K1: temperature from enthalpy by Newton on NASA-7 (NS (1)).
//
// HBM-bound: 4(K+2) bytes in + 4 (T) [+ 4 (cp)] out per cell.  One thread owns 4 consecutive cells
// (float4 SoA loads, coalesced across the warp).  For fixed Y, h(T,Y) is itself one polynomial in
// tau = (T - T_mid)/S with mixture coefficients C_m = sum_k Y_k c_{k,m}: the K-loop runs once
// (12 FMAs per species per cell, both ranges), every Newton iteration is then K-independent.
// fp32 iterations bring T to within a few mK; one fp64 Newton step on the species-level
// polynomials (fp64 tables, the selected range only) removes the fp32 cancellation error.
#include "common.cuh"

namespace {

constexpr int kThreads = 128;
constexpr int kMaxIter = 24;

__global__ void __launch_bounds__(kThreads)
t_from_h_kernel(int K, MechScalars sc, const float* __restrict__ th32, const double* __restrict__ th64,
                long long n, long long ld, const float* __restrict__ h, const float* __restrict__ Y,
                float* __restrict__ T, float* __restrict__ cp_out, int* __restrict__ n_unconv) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* s64 = reinterpret_cast<double*>(smem_raw);              // [K][2][6]
    float* s32 = reinterpret_cast<float*>(smem_raw + (size_t)K * 12 * sizeof(double));  // [K][12]
    for (int i = threadIdx.x; i < K * 12; i += kThreads) {
        s64[i] = th64[i];
        s32[i] = th32[i];
    }
    __syncthreads();

    const long long i0 = ((long long)blockIdx.x * kThreads + threadIdx.x) * 4;
    if (i0 >= n) return;
    const bool full = (i0 + 4 <= n);

    // ---- one pass over species: mixture polynomial coefficients, both ranges -----------------
    float C[4][12];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int m = 0; m < 12; ++m) C[c][m] = 0.f;

#pragma unroll 4
    for (int k = 0; k < K; ++k) {
        float y[4];
        const float* yp = Y + (size_t)k * ld + i0;
        if (full) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(yp));
            y[0] = v.x; y[1] = v.y; y[2] = v.z; y[3] = v.w;
        } else {
#pragma unroll
            for (int c = 0; c < 4; ++c) y[c] = (i0 + c < n) ? yp[c] : 0.f;
        }
        const float4* cf = reinterpret_cast<const float4*>(s32 + k * 12);
        const float4 a = cf[0], b = cf[1], d = cf[2];
        const float co[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, d.x, d.y, d.z, d.w};
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int m = 0; m < 12; ++m) C[c][m] = fmaf(y[c], co[m], C[c][m]);
    }

    float hin[4], tg[4];
    if (full) {
        const float4 hv = __ldg(reinterpret_cast<const float4*>(h + i0));
        const float4 tv = *reinterpret_cast<const float4*>(T + i0);
        hin[0] = hv.x; hin[1] = hv.y; hin[2] = hv.z; hin[3] = hv.w;
        tg[0] = tv.x; tg[1] = tv.y; tg[2] = tv.z; tg[3] = tv.w;
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            hin[c] = (i0 + c < n) ? h[i0 + c] : 0.f;
            tg[c] = (i0 + c < n) ? T[i0 + c] : 0.f;
        }
    }

    float Tout[4], cpv[4];
    int bad = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const bool live = (i0 + c < n);
        // A4: invalid guess -> T_mid (tau = 0)
        float tau = (tg[c] > 0.f && tg[c] < 3.0e38f) ? (tg[c] - sc.T_mid) * sc.inv_S : 0.f;
        tau = fminf(fmaxf(tau, sc.tau_min), sc.tau_max);
        float dh = 1.f;
        if (live) {
            for (int it = 0; it < kMaxIter; ++it) {
                const bool lo = tau < 0.f;  // register selects: a pointer would push C[][] to local memory
                const float q0 = lo ? C[c][0] : C[c][6], q1 = lo ? C[c][1] : C[c][7], q2 = lo ? C[c][2] : C[c][8],
                            q3 = lo ? C[c][3] : C[c][9], q4 = lo ? C[c][4] : C[c][10], q5 = lo ? C[c][5] : C[c][11];
                const float hv = fmaf(fmaf(fmaf(fmaf(fmaf(q5, tau, q4), tau, q3), tau, q2), tau, q1), tau, q0);
                dh = fmaf(fmaf(fmaf(fmaf(5.f * q5, tau, 4.f * q4), tau, 3.f * q3), tau, 2.f * q2), tau, q1);
                const float delta = (hin[c] - hv) / dh;
                tau = fminf(fmaxf(tau + delta, sc.tau_min), sc.tau_max);
                if (fabsf(delta) < 1e-5f) break;  // 10 mK: above the fp32 noise floor of h; the polish does the rest
            }
        }
        // ---- fp64 polish on the species-level polynomials of the selected range ---------------
        const int r = (tau < 0.f) ? 0 : 1;
        const double t = (double)tau;
        double hv = 0.0;
        if (live) {
            for (int k = 0; k < K; ++k) {
                const double* q = s64 + (k * 2 + r) * 6;
                const double pk = fma(fma(fma(fma(fma(q[5], t, q[4]), t, q[3]), t, q[2]), t, q[1]), t, q[0]);
                hv = fma((double)__ldg(Y + (size_t)k * ld + i0 + c), pk, hv);
            }
        }
        {
            const float q1 = r ? C[c][7] : C[c][1], q2 = r ? C[c][8] : C[c][2], q3 = r ? C[c][9] : C[c][3],
                        q4 = r ? C[c][10] : C[c][4], q5 = r ? C[c][11] : C[c][5];
            dh = fmaf(fmaf(fmaf(fmaf(5.f * q5, tau, 4.f * q4), tau, 3.f * q3), tau, 2.f * q2), tau, q1);
        }
        const double delta = live ? ((double)hin[c] - hv) / (double)dh : 0.0;
        double t2 = t + delta;
        t2 = fmin(fmax(t2, (double)sc.tau_min), (double)sc.tau_max);
        Tout[c] = (float)fma(t2, (double)sc.S, (double)sc.T_mid);
        // cp at the solution (range by the polished tau, A2)
        {
            const float tf = (float)t2;
            const bool lo = tf < 0.f;
            const float q1 = lo ? C[c][1] : C[c][7], q2 = lo ? C[c][2] : C[c][8], q3 = lo ? C[c][3] : C[c][9],
                        q4 = lo ? C[c][4] : C[c][10], q5 = lo ? C[c][5] : C[c][11];
            cpv[c] = fmaf(fmaf(fmaf(fmaf(5.f * q5, tf, 4.f * q4), tf, 3.f * q3), tf, 2.f * q2), tf, q1) * sc.inv_S;
        }
        if (live && !(fabs(delta) * (double)sc.S <= 1e-2)) ++bad;
    }

    if (full) {
        *reinterpret_cast<float4*>(T + i0) = make_float4(Tout[0], Tout[1], Tout[2], Tout[3]);
        if (cp_out) *reinterpret_cast<float4*>(cp_out + i0) = make_float4(cpv[0], cpv[1], cpv[2], cpv[3]);
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (i0 + c < n) {
                T[i0 + c] = Tout[c];
                if (cp_out) cp_out[i0 + c] = cpv[c];
            }
    }
    if (n_unconv && bad) atomicAdd(n_unconv, bad);
}

}  // namespace

df_status launch_T_from_h(const df_mech* mech, long long n, long long ld, const float* h, const float* Y, float* T,
                          float* cp, int* n_unconv, cudaStream_t s) {
    const int K = mech->K;
    const size_t smem = (size_t)K * 12 * (sizeof(double) + sizeof(float));
    const long long per_block = (long long)kThreads * 4;
    const long long blocks = (n + per_block - 1) / per_block;
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_T_from_h: n_cells too large");
    t_from_h_kernel<<<(unsigned)blocks, kThreads, smem, s>>>(K, mech->dev.sc, mech->dev.th32, mech->dev.th64, n, ld, h,
                                                            Y, T, cp, n_unconv);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

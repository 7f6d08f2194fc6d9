// t_from_h.cu -- K1: temperature from enthalpy by Newton on NASA-7 (NS (1)).
//
// HBM-bound: 4(K+2) bytes in + 4 (T) [+ 4 (cp)] out per cell.  One thread owns 4 consecutive cells
// (float4 SoA loads, coalesced across the warp).  For fixed Y, h(T,Y) is itself one polynomial in
// tau = (T - T_mid)/S with mixture coefficients C_m = sum_k Y_k c_{k,m}: the K-loop runs once
// (12 FMAs per species per cell, both ranges), every Newton iteration is then K-independent.
// fp32 iterations bring T to within a few mK; one fp64 Newton step on the species-level
// polynomials (fp64 tables, the selected range only) removes the fp32 cancellation error.
#include "common.cuh"
#include <cstdlib>

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


// ---- fixed K: two cells per thread, every load issued before the first use ---------------------------------------
// The generic kernel above alternates a load phase (4 float4 loads in flight per thread) with a long per-cell
// Newton / fp64 phase and re-reads Y for the fp64 step; it sustains ~2 TB/s.  For the species counts of the configs
// the whole column of Y (K float2 per thread) fits in registers: all K loads are in flight at once (3x the bytes in
// flight per SM) and the fp64 step needs no second pass.
#ifndef DF_TFH_MINBLOCKS
#define DF_TFH_MINBLOCKS 5
#endif
template <int K>
__global__ void __launch_bounds__(kThreads, DF_TFH_MINBLOCKS)
t_from_h_fixed_kernel(MechScalars sc, const float* __restrict__ th32, const double* __restrict__ th64, long long n,
                      long long ld, const float* __restrict__ h, const float* __restrict__ Y, float* __restrict__ T,
                      float* __restrict__ cp_out, int* __restrict__ n_unconv) {
    __shared__ __align__(16) double s64[K * 12];
    __shared__ __align__(16) float s32[K * 12];
    const long long i0 = ((long long)blockIdx.x * kThreads + threadIdx.x) * 2;
    const bool any = i0 < n, two = i0 + 1 < n;
    const long long ic = any ? i0 : 0;
    // the field loads go out first; the table staging below overlaps with their latency
    float2 y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const float* yp = Y + (size_t)k * ld + ic;
        if (two) y[k] = __ldg(reinterpret_cast<const float2*>(yp));
        else { const float v = __ldg(yp); y[k] = make_float2(v, v); }
    }
    float2 hin, tg;
    if (two) { hin = __ldg(reinterpret_cast<const float2*>(h + ic)); tg = *reinterpret_cast<const float2*>(T + ic); }
    else { hin = make_float2(__ldg(h + ic), 0.f); hin.y = hin.x; tg = make_float2(T[ic], T[ic]); }
    for (int i = threadIdx.x; i < K * 12; i += kThreads) {
        s64[i] = th64[i];
        s32[i] = th32[i];
    }
    __syncthreads();
    if (!any) return;

    // mixture polynomial coefficients, both ranges, both cells packed (FFMA2, coefficient broadcast)
    float2 P[12];
#pragma unroll
    for (int m = 0; m < 12; ++m) P[m] = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const float4* cf = reinterpret_cast<const float4*>(s32 + k * 12);
        const float4 a = cf[0], b = cf[1], d = cf[2];
        const float co[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, d.x, d.y, d.z, d.w};
#pragma unroll
        for (int m = 0; m < 12; ++m) P[m] = __ffma2_rn(y[k], make_float2(co[m], co[m]), P[m]);
    }
    float tauv[2], Tout[2], cpv[2];
    const float hv[2] = {hin.x, hin.y}, tgv[2] = {tg.x, tg.y};
    int bad = 0;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        float C[12];
#pragma unroll
        for (int m = 0; m < 12; ++m) C[m] = c ? P[m].y : P[m].x;
        float tau = (tgv[c] > 0.f && tgv[c] < 3.0e38f) ? (tgv[c] - sc.T_mid) * sc.inv_S : 0.f;  // A4
        tau = fminf(fmaxf(tau, sc.tau_min), sc.tau_max);
        for (int it = 0; it < kMaxIter; ++it) {
            const bool lo = tau < 0.f;
            const float q0 = lo ? C[0] : C[6], q1 = lo ? C[1] : C[7], q2 = lo ? C[2] : C[8], q3 = lo ? C[3] : C[9],
                        q4 = lo ? C[4] : C[10], q5 = lo ? C[5] : C[11];
            const float hh = fmaf(fmaf(fmaf(fmaf(fmaf(q5, tau, q4), tau, q3), tau, q2), tau, q1), tau, q0);
            const float dh = fmaf(fmaf(fmaf(fmaf(5.f * q5, tau, 4.f * q4), tau, 3.f * q3), tau, 2.f * q2), tau, q1);
            const float delta = (hv[c] - hh) / dh;
            tau = fminf(fmaxf(tau + delta, sc.tau_min), sc.tau_max);
            if (fabsf(delta) < 1e-5f) break;  // 10 mK: above the fp32 noise floor of h; the fp64 step does the rest
        }
        tauv[c] = tau;
    }
    // one fp64 Newton step on the species-level polynomials (Y still in registers), the two cells interleaved
    const int r0 = tauv[0] < 0.f ? 0 : 6, r1 = tauv[1] < 0.f ? 0 : 6;
    const double t0 = (double)tauv[0], t1 = (double)tauv[1];
    double h0 = 0.0, h1 = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const double* q0 = s64 + k * 12 + r0;
        const double* q1 = s64 + k * 12 + r1;
        const double p0 = fma(fma(fma(fma(fma(q0[5], t0, q0[4]), t0, q0[3]), t0, q0[2]), t0, q0[1]), t0, q0[0]);
        const double p1 = fma(fma(fma(fma(fma(q1[5], t1, q1[4]), t1, q1[3]), t1, q1[2]), t1, q1[1]), t1, q1[0]);
        h0 = fma((double)y[k].x, p0, h0);
        h1 = fma((double)y[k].y, p1, h1);
    }
    const double hv64[2] = {h0, h1};
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const float tau = tauv[c];
        const bool hi = !(tau < 0.f);
        const float q1 = c ? (hi ? P[7].y : P[1].y) : (hi ? P[7].x : P[1].x), q2 = c ? (hi ? P[8].y : P[2].y) : (hi ? P[8].x : P[2].x),
                    q3 = c ? (hi ? P[9].y : P[3].y) : (hi ? P[9].x : P[3].x), q4 = c ? (hi ? P[10].y : P[4].y) : (hi ? P[10].x : P[4].x),
                    q5 = c ? (hi ? P[11].y : P[5].y) : (hi ? P[11].x : P[5].x);
        const float dh = fmaf(fmaf(fmaf(fmaf(5.f * q5, tau, 4.f * q4), tau, 3.f * q3), tau, 2.f * q2), tau, q1);
        const double delta = ((double)hv[c] - hv64[c]) / (double)dh;
        double t2 = (double)tau + delta;
        t2 = fmin(fmax(t2, (double)sc.tau_min), (double)sc.tau_max);
        Tout[c] = (float)fma(t2, (double)sc.S, (double)sc.T_mid);
        const float tf = (float)t2;
        const bool lo = tf < 0.f;  // cp at the solution: range by the polished tau (A2)
        const float p1 = c ? (lo ? P[1].y : P[7].y) : (lo ? P[1].x : P[7].x), p2 = c ? (lo ? P[2].y : P[8].y) : (lo ? P[2].x : P[8].x),
                    p3 = c ? (lo ? P[3].y : P[9].y) : (lo ? P[3].x : P[9].x), p4 = c ? (lo ? P[4].y : P[10].y) : (lo ? P[4].x : P[10].x),
                    p5 = c ? (lo ? P[5].y : P[11].y) : (lo ? P[5].x : P[11].x);
        cpv[c] = fmaf(fmaf(fmaf(fmaf(5.f * p5, tf, 4.f * p4), tf, 3.f * p3), tf, 2.f * p2), tf, p1) * sc.inv_S;
        if ((c == 0 || two) && !(fabs(delta) * (double)sc.S <= 1e-2)) ++bad;
    }
    if (two) {
        *reinterpret_cast<float2*>(T + i0) = make_float2(Tout[0], Tout[1]);
        if (cp_out) *reinterpret_cast<float2*>(cp_out + i0) = make_float2(cpv[0], cpv[1]);
    } else {
        T[i0] = Tout[0];
        if (cp_out) cp_out[i0] = cpv[0];
    }
    if (n_unconv && bad) atomicAdd(n_unconv, bad);
}


// ---- fixed K, all-fp64 solve: one range per cell, no fp32 pass --------------------------------------------------
// h(T, Y) is increasing in T and both ranges agree at T_mid, so the side of the root is known before any iteration:
// hi iff h_in >= h(T_mid, Y) = sum_k Y_k c_{k,0} (an fp32 sum is enough: a cell within ~1 mK of T_mid may take either
// polynomial, they match there to second derivative).  Only the selected range's six mixture coefficients are then
// accumulated, in fp64 straight from the fp64 tables (6K DFMA per cell), and Newton runs in fp64 on that one
// polynomial (5 DFMA per iteration; the slope and its reciprocal in fp32 -- a quasi-Newton step with a 1e-7 relative
// slope error still contracts the error by 1e-7 per iteration).  Against the fp32-pass + fp64-polish kernel above:
// no 12K packed FMAs, no fp32 Newton with range selects, same number of fp64 operations.
template <int K>
__global__ void __launch_bounds__(kThreads, DF_TFH_MINBLOCKS)
t_from_h_f64_kernel(MechScalars sc, const float* __restrict__ th32, const double* __restrict__ th64, long long n,
                    long long ld, const float* __restrict__ h, const float* __restrict__ Y, float* __restrict__ T,
                    float* __restrict__ cp_out, int* __restrict__ n_unconv) {
    __shared__ __align__(16) double s64[K * 12];
    __shared__ __align__(16) float s0[(K + 3) & ~3];
    const long long i0 = ((long long)blockIdx.x * kThreads + threadIdx.x) * 2;
    const bool any = i0 < n, two = i0 + 1 < n;
    const long long ic = any ? i0 : 0;
    float2 y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const float* yp = Y + (size_t)k * ld + ic;
        if (two) y[k] = __ldg(reinterpret_cast<const float2*>(yp));
        else { const float v = __ldg(yp); y[k] = make_float2(v, v); }
    }
    float2 hin, tg;
    if (two) { hin = __ldg(reinterpret_cast<const float2*>(h + ic)); tg = *reinterpret_cast<const float2*>(T + ic); }
    else { hin = make_float2(__ldg(h + ic), 0.f); hin.y = hin.x; tg = make_float2(T[ic], T[ic]); }
    for (int i = threadIdx.x; i < K * 12; i += kThreads) s64[i] = th64[i];
    if (threadIdx.x < K) s0[threadIdx.x] = th32[threadIdx.x * 12 + 6];
    __syncthreads();
    if (!any) return;

    float2 hm = make_float2(0.f, 0.f);  // h(T_mid, Y), both cells
#pragma unroll
    for (int k = 0; k < K; ++k) hm = __ffma2_rn(y[k], make_float2(s0[k], s0[k]), hm);
    const bool hi0 = !(hin.x < hm.x), hi1 = !(hin.y < hm.y);  // A2: hi for T >= T_mid
    const double* qa = s64 + (hi0 ? 6 : 0);
    const double* qb = s64 + (hi1 ? 6 : 0);
    double A[6], Bc[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) A[m] = Bc[m] = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const double ya = (double)y[k].x, yb = (double)y[k].y;
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            A[m] = fma(ya, qa[k * 12 + m], A[m]);
            Bc[m] = fma(yb, qb[k * 12 + m], Bc[m]);
        }
    }
    // slope coefficients in fp32
    const float a1 = (float)A[1], a2 = 2.f * (float)A[2], a3 = 3.f * (float)A[3], a4 = 4.f * (float)A[4], a5 = 5.f * (float)A[5];
    const float b1 = (float)Bc[1], b2 = 2.f * (float)Bc[2], b3 = 3.f * (float)Bc[3], b4 = 4.f * (float)Bc[4], b5 = 5.f * (float)Bc[5];
    // A4: invalid guess -> T_mid; the start is moved onto the root's side of T_mid, the iterates stay there
    float ga = (tg.x > 0.f && tg.x < 3.0e38f) ? (tg.x - sc.T_mid) * sc.inv_S : 0.f;
    float gb = (tg.y > 0.f && tg.y < 3.0e38f) ? (tg.y - sc.T_mid) * sc.inv_S : 0.f;
    const double la = hi0 ? 0.0 : (double)sc.tau_min, ua = hi0 ? (double)sc.tau_max : 0.0;
    const double lb = hi1 ? 0.0 : (double)sc.tau_min, ub = hi1 ? (double)sc.tau_max : 0.0;
    double ta = fmin(fmax((double)ga, la), ua), tb = fmin(fmax((double)gb, lb), ub);
    const double ha = (double)hin.x, hb = (double)hin.y;
    double da = 0.0, db = 0.0;
    for (int it = 0; it < kMaxIter; ++it) {
        const double va = fma(fma(fma(fma(fma(A[5], ta, A[4]), ta, A[3]), ta, A[2]), ta, A[1]), ta, A[0]);
        const double vb = fma(fma(fma(fma(fma(Bc[5], tb, Bc[4]), tb, Bc[3]), tb, Bc[2]), tb, Bc[1]), tb, Bc[0]);
        const float fa = (float)ta, fb = (float)tb;
        const float sa = fmaf(fmaf(fmaf(fmaf(a5, fa, a4), fa, a3), fa, a2), fa, a1);
        const float sb = fmaf(fmaf(fmaf(fmaf(b5, fb, b4), fb, b3), fb, b2), fb, b1);
        da = (ha - va) * (double)__frcp_rn(sa);
        db = (hb - vb) * (double)__frcp_rn(sb);
        ta = fmin(fmax(ta + da, la), ua);
        tb = fmin(fmax(tb + db, lb), ub);
        if (!(fmax(fabs(da), fabs(db)) >= 1e-6)) break;  // 1 mK step: the error left is ~1e-9 K (also leaves on NaN)
    }
    const float fa = (float)ta, fb = (float)tb;
    const float cpa = fmaf(fmaf(fmaf(fmaf(a5, fa, a4), fa, a3), fa, a2), fa, a1) * sc.inv_S;
    const float cpb = fmaf(fmaf(fmaf(fmaf(b5, fb, b4), fb, b3), fb, b2), fb, b1) * sc.inv_S;
    const float Ta = (float)fma(ta, (double)sc.S, (double)sc.T_mid), Tb = (float)fma(tb, (double)sc.S, (double)sc.T_mid);
    int bad = 0;
    if (!(fabs(da) * (double)sc.S <= 1e-2)) ++bad;
    if (two && !(fabs(db) * (double)sc.S <= 1e-2)) ++bad;
    if (two) {
        *reinterpret_cast<float2*>(T + i0) = make_float2(Ta, Tb);
        if (cp_out) *reinterpret_cast<float2*>(cp_out + i0) = make_float2(cpa, cpb);
    } else {
        T[i0] = Ta;
        if (cp_out) cp_out[i0] = cpa;
    }
    if (n_unconv && bad) atomicAdd(n_unconv, bad);
}

template <int K>
df_status launch_fixed(const df_mech* mech, long long n, long long ld, const float* h, const float* Y, float* T, float* cp,
                       int* n_unconv, cudaStream_t s) {
    const long long blocks = (n + 2 * kThreads - 1) / (2 * kThreads);
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_T_from_h: n_cells too large");
    static const bool v1 = getenv("DF_TFH_V1") != nullptr;
    if (v1)
        t_from_h_fixed_kernel<K><<<(unsigned)blocks, kThreads, 0, s>>>(mech->dev.sc, mech->dev.th32, mech->dev.th64, n, ld, h, Y,
                                                                       T, cp, n_unconv);
    else
        t_from_h_f64_kernel<K><<<(unsigned)blocks, kThreads, 0, s>>>(mech->dev.sc, mech->dev.th32, mech->dev.th64, n, ld, h, Y,
                                                                     T, cp, n_unconv);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

}  // namespace

df_status launch_T_from_h(const df_mech* mech, long long n, long long ld, const float* h, const float* Y, float* T,
                          float* cp, int* n_unconv, cudaStream_t s) {
    const int K = mech->K;
    if (K == 19) return launch_fixed<19>(mech, n, ld, h, Y, T, cp, n_unconv, s);
    if (K == 9) return launch_fixed<9>(mech, n, ld, h, Y, T, cp, n_unconv, s);
    const size_t smem = (size_t)K * 12 * (sizeof(double) + sizeof(float));
    const long long per_block = (long long)kThreads * 4;
    const long long blocks = (n + per_block - 1) / per_block;
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_T_from_h: n_cells too large");
    t_from_h_kernel<<<(unsigned)blocks, kThreads, smem, s>>>(K, mech->dev.sc, mech->dev.th32, mech->dev.th64, n, ld, h,
                                                            Y, T, cp, n_unconv);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

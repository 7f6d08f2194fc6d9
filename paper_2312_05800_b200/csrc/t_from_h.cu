// t_from_h.cu -- K1: temperature from enthalpy by Newton on NASA-7 (NS (1)).
//
// HBM-bound: 4(K+2) bytes in + 4 (T) [+ 4 (cp)] out per cell.  For fixed Y, h(T,Y) is itself one polynomial in
// tau = (T - T_mid)/S with mixture coefficients C_m = sum_k Y_k c_{k,m}: the K-loop runs once, every Newton
// iteration is then K-independent.  Two kernels:
//  * t_from_h_sorted_kernel<K> (K = 9, 19: the configs' species counts): all fp64, one range per cell, the block's
//    cells sorted by range through shared memory so that the table reads are warp-uniform (see its header below);
//  * t_from_h_kernel (any K): one thread owns 4 consecutive cells (float4 SoA loads); fp32 mixture coefficients of
//    both ranges (12 FMAs per species per cell), fp32 iterations to a few mK, then one fp64 Newton step on the
//    species-level polynomials (fp64 tables, the selected range only) that removes the fp32 cancellation error.
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


// ---- fixed K: all-fp64 solve on range-sorted blocks ----------------------------------------------------------------
// h(T, Y) is increasing in T and both ranges agree at T_mid, so the side of the root is known before any iteration:
// hi iff h_in >= h(T_mid, Y) = sum_k Y_k c_{k,0} (an fp32 sum is enough: a cell within ~1 mK of T_mid may take either
// polynomial, they match there).  Only that range's six mixture coefficients are accumulated, in fp64 straight from
// the fp64 tables (6K DFMA per cell), and Newton runs in fp64 on that one polynomial (5 DFMA per iteration; slope and
// reciprocal in fp32: a quasi-Newton step with a 1e-7 relative slope error still contracts the error by 1e-7).
//
// The coefficient pass is bound by shared-memory wavefronts, not by the fp64 pipe: with per-lane table addresses
// (each lane its own range) every LDS.128 is a four-wavefront access -- 912 B of coefficients per cell through the
// 128 B/clk return path is 7 clk per cell per SM against the 2 clk per cell HBM needs (measured on config 5:
// 0.515 ms with per-lane ranges, 0.37 ms with one range forced).  So the block first sorts its 256 cells by range
// through shared memory (hi cells from slot 0 up, lo cells from slot 255 down), after which at most one of its four
// warps holds both ranges; the others read the tables at compile-time addresses (broadcast: one wavefront).  The one
// mixed warp reads both ranges, also at uniform addresses, and feeds each cell's Y into its own range's sum (the other
// range gets 0): twice the DFMAs for a quarter of the warps instead of four times the wavefronts.  A thread loads
// cells t and t + 128 of the block, so that the lanes of a warp scatter to consecutive slots (few bank conflicts),
// and owns the adjacent slots 2t, 2t + 1 afterwards.  Results go back through shared memory to their own cells: the
// global stores stay coalesced.
constexpr int kSCells = 2 * kThreads;
#ifndef DF_TFH_MINBLOCKS
#define DF_TFH_MINBLOCKS 5
#endif

template <int K>
__device__ __forceinline__ void mixture_coeffs(const float2 (&y)[K], const double* q, double (&A)[6], double (&Bc)[6]) {
#pragma unroll
    for (int m = 0; m < 6; ++m) A[m] = Bc[m] = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const double ya = (double)y[k].x, yb = (double)y[k].y;
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            A[m] = fma(ya, q[k * 12 + m], A[m]);
            Bc[m] = fma(yb, q[k * 12 + m], Bc[m]);
        }
    }
}

template <int K>
__device__ __forceinline__ void mixture_coeffs_mixed(const float2 (&y)[K], const double* s64, bool hi_a, bool hi_b,
                                                     double (&A)[6], double (&Bc)[6]) {
#pragma unroll
    for (int m = 0; m < 6; ++m) A[m] = Bc[m] = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const double ya = (double)y[k].x, yb = (double)y[k].y;
        const double ya_hi = hi_a ? ya : 0.0, ya_lo = hi_a ? 0.0 : ya, yb_hi = hi_b ? yb : 0.0, yb_lo = hi_b ? 0.0 : yb;
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            const double lo = s64[k * 12 + m], hi = s64[k * 12 + 6 + m];
            A[m] = fma(ya_hi, hi, fma(ya_lo, lo, A[m]));
            Bc[m] = fma(yb_hi, hi, fma(yb_lo, lo, Bc[m]));
        }
    }
}

template <int K>
constexpr size_t sorted_smem_bytes() {
    return (size_t)K * 12 * sizeof(double) + ((size_t)(K + 2) * kSCells + 2 * kSCells + ((K + 3) & ~3) + 8) * sizeof(float) +
           kSCells * sizeof(unsigned short);
}

template <int K>
__global__ void __launch_bounds__(kThreads, DF_TFH_MINBLOCKS)
t_from_h_sorted_kernel(MechScalars sc, const float* __restrict__ th32, const double* __restrict__ th64, long long n,
                       long long ld, const float* __restrict__ h, const float* __restrict__ Y, float* __restrict__ T,
                       float* __restrict__ cp_out, int* __restrict__ n_unconv) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* s64 = reinterpret_cast<double*>(smem_raw);                  // [K][2][6]
    float* buf = reinterpret_cast<float*>(smem_raw + (size_t)K * 96);   // [K + 2][256]: Y rows, h, guess (sorted slots)
    float* out = buf + (K + 2) * kSCells;                               // [2][256]: T, cp (own cells)
    float* s0 = out + 2 * kSCells;                                      // h_k(T_mid)
    int* wcount = reinterpret_cast<int*>(s0 + ((K + 3) & ~3));          // hi cells per (half, warp)
    unsigned short* orig = reinterpret_cast<unsigned short*>(wcount + 8);  // slot -> cell of the block

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long base = (long long)blockIdx.x * kSCells;
    const int c0 = tid, c1 = tid + kThreads;  // this thread's cells before the sort
    const bool in0 = base + c0 < n, in1 = base + c1 < n;
    const long long i0 = in0 ? base + c0 : 0, i1 = in1 ? base + c1 : 0;
    float2 y[K], hin, tg;
    if (base + kSCells <= n) {  // whole block in range: one pointer, the second cell at a constant offset
        const float* yp = Y + i0;
#pragma unroll
        for (int k = 0; k < K; ++k, yp += ld) y[k] = make_float2(__ldg(yp), __ldg(yp + kThreads));
        hin = make_float2(__ldg(h + i0), __ldg(h + i0 + kThreads));
        tg = make_float2(T[i0], T[i0 + kThreads]);
    } else {
#pragma unroll
        for (int k = 0; k < K; ++k) y[k] = make_float2(__ldg(Y + (size_t)k * ld + i0), __ldg(Y + (size_t)k * ld + i1));
        hin = make_float2(__ldg(h + i0), __ldg(h + i1));
        tg = make_float2(T[i0], T[i1]);
    }
    for (int i = tid; i < K * 12; i += kThreads) s64[i] = th64[i];
    if (tid < K) s0[tid] = th32[tid * 12 + 6];
    __syncthreads();

    // side of the root: hi iff h_in >= h(T_mid, Y) (A2); cells past n count as lo
    float2 hm = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < K; ++k) hm = __ffma2_rn(y[k], make_float2(s0[k], s0[k]), hm);
    const bool hi0 = in0 && !(hin.x < hm.x), hi1 = in1 && !(hin.y < hm.y);
    const unsigned m0 = __ballot_sync(0xffffffffu, hi0), m1 = __ballot_sync(0xffffffffu, hi1);
    const unsigned lt = (1u << lane) - 1u;
    if (lane == 0) {
        wcount[warp] = __popc(m0);
        wcount[4 + warp] = __popc(m1);
    }
    __syncthreads();
    int before0 = __popc(m0 & lt), before1 = __popc(m1 & lt), tot = 0;  // hi cells ahead of c0 / c1 in cell order
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const int c = wcount[w];
        tot += c;
        if (w < warp) before0 += c;
        if (w < 4 + warp) before1 += c;
    }
    {
        const int sl0 = hi0 ? before0 : kSCells - 1 - (c0 - before0);
        const int sl1 = hi1 ? before1 : kSCells - 1 - (c1 - before1);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            buf[k * kSCells + sl0] = y[k].x;
            buf[k * kSCells + sl1] = y[k].y;
        }
        buf[K * kSCells + sl0] = hin.x;
        buf[K * kSCells + sl1] = hin.y;
        buf[(K + 1) * kSCells + sl0] = tg.x;
        buf[(K + 1) * kSCells + sl1] = tg.y;
        orig[sl0] = (unsigned short)c0;
        orig[sl1] = (unsigned short)c1;
    }
    __syncthreads();
    const int p0 = 2 * tid;  // this thread's slots after the sort
#pragma unroll
    for (int k = 0; k < K; ++k) y[k] = *reinterpret_cast<const float2*>(buf + k * kSCells + p0);
    hin = *reinterpret_cast<const float2*>(buf + K * kSCells + p0);
    tg = *reinterpret_cast<const float2*>(buf + (K + 1) * kSCells + p0);
    const int o0 = orig[p0], o1 = orig[p0 + 1];
    const bool v0 = base + o0 < n, v1 = base + o1 < n;
    const bool s_hi0 = p0 < tot, s_hi1 = p0 + 1 < tot;

    double A[6], Bc[6];
    if (warp * 64 + 64 <= tot) mixture_coeffs<K>(y, s64 + 6, A, Bc);
    else if (warp * 64 >= tot) mixture_coeffs<K>(y, s64, A, Bc);
    else mixture_coeffs_mixed<K>(y, s64, s_hi0, s_hi1, A, Bc);

    // slope coefficients in fp32
    const float a1 = (float)A[1], a2 = 2.f * (float)A[2], a3 = 3.f * (float)A[3], a4 = 4.f * (float)A[4], a5 = 5.f * (float)A[5];
    const float b1 = (float)Bc[1], b2 = 2.f * (float)Bc[2], b3 = 3.f * (float)Bc[3], b4 = 4.f * (float)Bc[4], b5 = 5.f * (float)Bc[5];
    // A4: invalid guess -> T_mid; the start is moved onto the root's side of T_mid, the iterates stay there
    const float ga = (tg.x > 0.f && tg.x < 3.0e38f) ? (tg.x - sc.T_mid) * sc.inv_S : 0.f;
    const float gb = (tg.y > 0.f && tg.y < 3.0e38f) ? (tg.y - sc.T_mid) * sc.inv_S : 0.f;
    // (the side was picked in fp32: a root within a few mK of T_mid may lie just across it, hence the 1 K margin)
    constexpr double kMargin = 1e-3;
    const double la = s_hi0 ? -kMargin : (double)sc.tau_min, ua = s_hi0 ? (double)sc.tau_max : kMargin;
    const double lb = s_hi1 ? -kMargin : (double)sc.tau_min, ub = s_hi1 ? (double)sc.tau_max : kMargin;
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
    out[o0] = (float)fma(ta, (double)sc.S, (double)sc.T_mid);
    out[o1] = (float)fma(tb, (double)sc.S, (double)sc.T_mid);
    out[kSCells + o0] = fmaf(fmaf(fmaf(fmaf(a5, fa, a4), fa, a3), fa, a2), fa, a1) * sc.inv_S;  // cp at the root
    out[kSCells + o1] = fmaf(fmaf(fmaf(fmaf(b5, fb, b4), fb, b3), fb, b2), fb, b1) * sc.inv_S;
    int bad = 0;
    if (v0 && !(fabs(da) * (double)sc.S <= 1e-2)) ++bad;
    if (v1 && !(fabs(db) * (double)sc.S <= 1e-2)) ++bad;
    if (n_unconv && bad) atomicAdd(n_unconv, bad);
    __syncthreads();
    if (in0) {
        T[base + c0] = out[c0];
        if (cp_out) cp_out[base + c0] = out[kSCells + c0];
    }
    if (in1) {
        T[base + c1] = out[c1];
        if (cp_out) cp_out[base + c1] = out[kSCells + c1];
    }
}

template <int K>
df_status launch_fixed(const df_mech* mech, long long n, long long ld, const float* h, const float* Y, float* T, float* cp,
                       int* n_unconv, cudaStream_t s) {
    const long long blocks = (n + kSCells - 1) / kSCells;
    if (blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_T_from_h: n_cells too large");
    static DfPerDevice smem_attr;
    const df_status st = df_ensure_dyn_smem((const void*)t_from_h_sorted_kernel<K>, (int)sorted_smem_bytes<K>(), &smem_attr);
    if (st != DF_OK) return st;
    t_from_h_sorted_kernel<K><<<(unsigned)blocks, kThreads, sorted_smem_bytes<K>(), s>>>(mech->dev.sc, mech->dev.th32,
                                                                                         mech->dev.th64, n, ld, h, Y, T, cp, n_unconv);
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

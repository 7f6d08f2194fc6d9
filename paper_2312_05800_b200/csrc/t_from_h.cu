// t_from_h.cu -- K1: temperature from enthalpy by Newton on NASA-7 (NS (1)).
//
// HBM-bound: 4(K+2) bytes in + 4 (T) [+ 4 (cp)] out per cell.  For fixed Y, h(T,Y) is itself one polynomial in
// tau = (T - T_mid)/S with mixture coefficients C_m = sum_k Y_k c_{k,m}: the K-loop runs once, every Newton
// iteration is then K-independent.  Two kernels:
//  * t_from_h_fixed_kernel<K> (K = 9, 19: the configs' species counts): fp64 coefficients of the high range for every
//    cell + an fp32 low-minus-high correction, tables in the constant bank, no shared memory (see its header below);
//  * t_from_h_kernel (any K): the same algorithm with the tables in shared memory and a run-time species loop.
// Both give a thread two adjacent cells (float2 SoA loads: 256 B per warp and species row).
#include "common.cuh"

namespace {

constexpr int kThreads = 128;
constexpr int kMaxIter = 24;

// Newton on the two cells of a thread once their mixture coefficients are known: A, Bc = high-range coefficients (fp64),
// d = packed low-minus-high corrections (fp32).  Returns the number of unconverged cells.
__device__ __forceinline__ int newton_pair(const MechScalars& sc, double (&A)[6], double (&Bc)[6], const float2 (&d)[6],
                                           float2 hin, float2 tg, bool two, float2& Tout, float2& cpv) {
    // side of the root (A2): hi iff h_in >= h(T_mid, Y); NaN counts as hi and leaves through the iteration cap
    const bool hi_a = !((double)hin.x < A[0]), hi_b = !((double)hin.y < Bc[0]);
    if (!hi_a) {
#pragma unroll
        for (int m = 0; m < 6; ++m) A[m] += (double)d[m].x;
    }
    if (!hi_b) {
#pragma unroll
        for (int m = 0; m < 6; ++m) Bc[m] += (double)d[m].y;
    }
    // slope coefficients in fp32
    const float a1 = (float)A[1], a2 = 2.f * (float)A[2], a3 = 3.f * (float)A[3], a4 = 4.f * (float)A[4], a5 = 5.f * (float)A[5];
    const float b1 = (float)Bc[1], b2 = 2.f * (float)Bc[2], b3 = 3.f * (float)Bc[3], b4 = 4.f * (float)Bc[4], b5 = 5.f * (float)Bc[5];
    // A4: invalid guess -> T_mid; the start is moved onto the root's side of T_mid, the iterates stay there
    // (a mechanism whose two ranges do not quite meet at T_mid may have its root a hair across it, hence the 1 K margin)
    constexpr float kMargin = 1e-3f;
    const float la = hi_a ? -kMargin : sc.tau_min, ua = hi_a ? sc.tau_max : kMargin;
    const float lb = hi_b ? -kMargin : sc.tau_min, ub = hi_b ? sc.tau_max : kMargin;
    const float ga = (tg.x > 0.f && tg.x < 3.0e38f) ? (tg.x - sc.T_mid) * sc.inv_S : 0.f;
    const float gb = (tg.y > 0.f && tg.y < 3.0e38f) ? (tg.y - sc.T_mid) * sc.inv_S : 0.f;
    double ta = (double)fminf(fmaxf(ga, la), ua), tb = (double)fminf(fmaxf(gb, lb), ub);
    const double ha = (double)hin.x, hb = (double)hin.y;
    // The residual is formed in fp64 (it is the difference of two numbers ~1e7 that must be good to 0.1); the step
    // itself -- residual x 1/slope -- needs no more than fp32: its rounding is 1e-7 of the step, a quasi-Newton
    // perturbation.  The loop leaves after a step below 10 mK: the error left is (step)^2 cp'/(2 cp) < 1e-7 K.
    float sa_step = 0.f, sb_step = 0.f;
    for (int it = 0; it < kMaxIter; ++it) {
        const double va = fma(fma(fma(fma(fma(A[5], ta, A[4]), ta, A[3]), ta, A[2]), ta, A[1]), ta, A[0]);
        const double vb = fma(fma(fma(fma(fma(Bc[5], tb, Bc[4]), tb, Bc[3]), tb, Bc[2]), tb, Bc[1]), tb, Bc[0]);
        const float fa = (float)ta, fb = (float)tb;
        const float sa = fmaf(fmaf(fmaf(fmaf(a5, fa, a4), fa, a3), fa, a2), fa, a1);
        const float sb = fmaf(fmaf(fmaf(fmaf(b5, fb, b4), fb, b3), fb, b2), fb, b1);
        sa_step = (float)(ha - va) * rcp_approx(sa);
        sb_step = (float)(hb - vb) * rcp_approx(sb);
        ta += (double)sa_step;
        tb += (double)sb_step;
        const float na = fa + sa_step, nb = fb + sb_step;   // where the iterate went, to fp32: enough for the (rare) clamp
        if (na < la) ta = (double)la;
        if (na > ua) ta = (double)ua;
        if (nb < lb) tb = (double)lb;
        if (nb > ub) tb = (double)ub;
        if (!(fmaxf(fabsf(sa_step), fabsf(sb_step)) >= 1e-5f)) break;   // also leaves on NaN
    }
    const float fa = (float)ta, fb = (float)tb;
    Tout = make_float2((float)fma(ta, (double)sc.S, (double)sc.T_mid), (float)fma(tb, (double)sc.S, (double)sc.T_mid));
    cpv = make_float2(fmaf(fmaf(fmaf(fmaf(a5, fa, a4), fa, a3), fa, a2), fa, a1) * sc.inv_S,   // cp at the root
                      fmaf(fmaf(fmaf(fmaf(b5, fb, b4), fb, b3), fb, b2), fb, b1) * sc.inv_S);
    int bad = 0;
    if (!(fabsf(sa_step) * sc.S <= 1e-2f)) ++bad;
    if (two && !(fabsf(sb_step) * sc.S <= 1e-2f)) ++bad;
    return bad;
}

// ---- fixed K (9, 19): fp64 coefficient pass without any range dependence ------------------------------------------
// h(T, Y) is increasing in T and both ranges agree at T_mid, so the side of the root is known before any iteration:
// hi iff h_in >= h(T_mid, Y).  The coefficient pass accumulates, for EVERY cell, the six mixture coefficients of the
// HIGH range in fp64 (6K DFMA per cell, tables in the constant bank: no shared memory, no sort, no barrier -- the
// round-1 kernel sorted each block's cells by range through shared memory to keep its table reads warp-uniform) and,
// packed in fp32 for the thread's two cells, the coefficients of the CORRECTION lo - hi (6K/2 FFMA2).  A low-range
// cell adds the correction to its coefficients once (E_m = A_m + d_m).  Why fp32 is enough there and nowhere else: the
// residual h(T) - h_in must be good to ~0.3 J/kg (1e-3 K x cp / 3) against |h| ~ 2e7 J/kg, i.e. 2e-8 relative; the
// correction, though, is the difference of two polynomials that agree to second order at T_mid, it is only ever
// evaluated on |tau| < 0.8, and its terms there are <~ 3e6 J/kg: their fp32 rounding is <~ 0.3 J/kg at 250 K and
// falls off as |tau|^3 towards T_mid (the opposite choice -- low range as the base -- would put the correction at
// tau = 2.5, 300x larger).  Newton then runs in fp64 on that one polynomial (5 DFMA per iteration; slope and
// reciprocal in fp32: a quasi-Newton step with a 1e-7 relative slope error still contracts the error by 1e-7).
template <int K>
struct TfhTables {
    double hi[K][6];    // h_k/W_k, high range, in tau
    float dlo[K][6];    // low range minus high range
    MechScalars sc;
};

// FULL: every thread has both of its cells inside the field (the ragged last block is launched separately): plain
// float2 accesses without the two-path predicates -- the kernel is issue-bound, every instruction counts.
template <int K, bool FULL>
__global__ void __launch_bounds__(kThreads, 6)
t_from_h_fixed_kernel(const __grid_constant__ TfhTables<K> tab, long long i_first, long long n, long long ld, const float* __restrict__ h,
                      const float* __restrict__ Y, float* __restrict__ T, float* __restrict__ cp_out, int* __restrict__ n_unconv) {
    const long long i = i_first + ((long long)blockIdx.x * kThreads + threadIdx.x) * 2;
    if (!FULL && i >= n) return;
    const bool two = FULL || i + 1 < n;   // ld % 4 == 0 and 16-byte aligned bases make the float2 accesses legal
    auto ld2 = [&](const float* p) -> float2 {
        if (two) return __ldg(reinterpret_cast<const float2*>(p + i));
        const float v = __ldg(p + i);
        return make_float2(v, v);
    };
    float2 y[K];
#pragma unroll
    for (int k = 0; k < K; ++k) y[k] = ld2(Y + (size_t)k * ld);
    const float2 hin = ld2(h);
    float2 tg;
    if (two) tg = *reinterpret_cast<const float2*>(T + i);
    else tg = make_float2(T[i], T[i]);
    const MechScalars& sc = tab.sc;

    double A[6], Bc[6];
    float2 d[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        A[m] = Bc[m] = 0.0;
        d[m] = make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const double ya = (double)y[k].x, yb = (double)y[k].y;
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            A[m] = fma(ya, tab.hi[k][m], A[m]);
            Bc[m] = fma(yb, tab.hi[k][m], Bc[m]);
            d[m] = __ffma2_rn(y[k], make_float2(tab.dlo[k][m], tab.dlo[k][m]), d[m]);
        }
    }
    float2 Tout, cpv;
    const int bad = newton_pair(sc, A, Bc, d, hin, tg, two, Tout, cpv);
    if (two) {
        *reinterpret_cast<float2*>(T + i) = Tout;
        if (cp_out) *reinterpret_cast<float2*>(cp_out + i) = cpv;
    } else {
        T[i] = Tout.x;
        if (cp_out) cp_out[i] = cpv.x;
    }
    if (n_unconv && bad) atomicAdd(n_unconv, bad);
}

template <int K>
df_status launch_fixed(const df_mech* mech, long long n, long long ld, const float* h, const float* Y, float* T, float* cp,
                       int* n_unconv, cudaStream_t s) {
    const long long full_blocks = n / (2 * kThreads), tail_first = full_blocks * 2 * kThreads;
    if (full_blocks > 0x7fffffffLL) return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_T_from_h: n_cells too large");
    TfhTables<K> tab;
    for (int k = 0; k < K; ++k)
        for (int m = 0; m < 6; ++m) {
            tab.hi[k][m] = mech->th64_host[(k * 2 + 1) * 6 + m];
            tab.dlo[k][m] = (float)(mech->th64_host[(k * 2) * 6 + m] - mech->th64_host[(k * 2 + 1) * 6 + m]);
        }
    tab.sc = mech->dev.sc;
    if (full_blocks > 0) t_from_h_fixed_kernel<K, true><<<(unsigned)full_blocks, kThreads, 0, s>>>(tab, 0, n, ld, h, Y, T, cp, n_unconv);
    if (tail_first < n) t_from_h_fixed_kernel<K, false><<<1, kThreads, 0, s>>>(tab, tail_first, n, ld, h, Y, T, cp, n_unconv);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

// ---- any K: the same algorithm with the tables in shared memory and a run-time species loop -----------------------
// A block stages the tables once and walks over tiles of 256 cells (grid-stride).  FULL: every tile of the launch lies
// inside the field (the host launches the ragged last tile separately): plain float2 accesses.
constexpr int kGenericBlocks = 6;   // resident blocks per SM (85 registers): 4 (126 registers) and 5 measured 9-13 % slower, 8 the same
template <bool FULL>
__global__ void __launch_bounds__(kThreads, kGenericBlocks)
t_from_h_kernel(int K, MechScalars sc, const double* __restrict__ th64, long long tile_first, long long tile_end, long long n,
                long long ld, const float* __restrict__ h, const float* __restrict__ Y, float* __restrict__ T,
                float* __restrict__ cp_out, int* __restrict__ n_unconv) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sHi = reinterpret_cast<double*>(smem_raw);                              // [K][6] high range
    float* sD = reinterpret_cast<float*>(smem_raw + (size_t)K * 6 * sizeof(double));   // [K][8] low - high (6 used)
    for (int e = threadIdx.x; e < K * 6; e += kThreads) {
        const int k = e / 6, m = e - 6 * k;
        const double hi = th64[(k * 2 + 1) * 6 + m];
        sHi[e] = hi;
        sD[k * 8 + m] = (float)(th64[(k * 2) * 6 + m] - hi);
    }
    __syncthreads();
    int bad = 0;
    for (long long tile = tile_first + blockIdx.x; tile < tile_end; tile += gridDim.x) {
        const long long i = (tile * kThreads + threadIdx.x) * 2;
        if (!FULL && i >= n) break;
        const bool two = FULL || i + 1 < n;
        auto ld2 = [&](const float* p) -> float2 {
            if (two) return __ldg(reinterpret_cast<const float2*>(p + i));
            const float v = __ldg(p + i);
            return make_float2(v, v);
        };
        double A[6], Bc[6];
        float2 d[6];
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            A[m] = Bc[m] = 0.0;
            d[m] = make_float2(0.f, 0.f);
        }
#pragma unroll 8
        for (int k = 0; k < K; ++k) {   // unrolled: eight rows of loads in flight per thread
            const float2 y = ld2(Y + (size_t)k * ld);
            const double ya = (double)y.x, yb = (double)y.y;
            const double2 h01 = *reinterpret_cast<const double2*>(sHi + k * 6), h23 = *reinterpret_cast<const double2*>(sHi + k * 6 + 2),
                          h45 = *reinterpret_cast<const double2*>(sHi + k * 6 + 4);
            const float4 d03 = *reinterpret_cast<const float4*>(sD + k * 8);
            const float2 d45 = *reinterpret_cast<const float2*>(sD + k * 8 + 4);
            const double hc[6] = {h01.x, h01.y, h23.x, h23.y, h45.x, h45.y};
            const float dc[6] = {d03.x, d03.y, d03.z, d03.w, d45.x, d45.y};
#pragma unroll
            for (int m = 0; m < 6; ++m) {
                A[m] = fma(ya, hc[m], A[m]);
                Bc[m] = fma(yb, hc[m], Bc[m]);
                d[m] = __ffma2_rn(y, make_float2(dc[m], dc[m]), d[m]);
            }
        }
        const float2 hin = ld2(h);
        float2 tg;
        if (two) tg = *reinterpret_cast<const float2*>(T + i);
        else tg = make_float2(T[i], T[i]);
        float2 Tout, cpv;
        bad += newton_pair(sc, A, Bc, d, hin, tg, two, Tout, cpv);
        if (two) {
            *reinterpret_cast<float2*>(T + i) = Tout;
            if (cp_out) *reinterpret_cast<float2*>(cp_out + i) = cpv;
        } else {
            T[i] = Tout.x;
            if (cp_out) cp_out[i] = cpv.x;
        }
    }
    if (n_unconv && bad) atomicAdd(n_unconv, bad);
}

}  // namespace

df_status launch_T_from_h(const df_mech* mech, long long n, long long ld, const float* h, const float* Y, float* T,
                          float* cp, int* n_unconv, cudaStream_t s) {
    const int K = mech->K;
    if (K == 19) return launch_fixed<19>(mech, n, ld, h, Y, T, cp, n_unconv, s);
    if (K == 9) return launch_fixed<9>(mech, n, ld, h, Y, T, cp, n_unconv, s);
    const size_t smem = (size_t)K * (6 * sizeof(double) + 8 * sizeof(float));
    const long long per_tile = (long long)kThreads * 2;
    const long long full_tiles = n / per_tile, tiles = (n + per_tile - 1) / per_tile;
    if (full_tiles > 0) {   // a few waves of resident blocks, each walking over its tiles
        const long long cap = (long long)df_device_sm_count() * kGenericBlocks * 8;
        const long long blocks = full_tiles < cap ? full_tiles : cap;
        t_from_h_kernel<true><<<(unsigned)blocks, kThreads, smem, s>>>(K, mech->dev.sc, mech->dev.th64, 0, full_tiles, n, ld, h, Y, T, cp, n_unconv);
    }
    if (tiles > full_tiles)
        t_from_h_kernel<false><<<1, kThreads, smem, s>>>(K, mech->dev.sc, mech->dev.th64, full_tiles, tiles, n, ld, h, Y, T, cp, n_unconv);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

// properties_group.cu -- K2 for any species count K <= 64 (BASELINE config 4: K = 53).  NS (2); A5-A7.
//
// At K = 53 the per-cell vectors (X, 1/g, S: 53 values each) do not fit in registers.  Kept per thread in shared
// memory they cap a thread-owns-its-cells kernel at 6 warps per SM (round 1: 26 % of the FP32 roofline, every
// O(K) phase exposed to global-memory latency).  Here FOUR WARPS SHARE ONE GROUP OF 64 CELLS: lane l of every warp
// holds cells 2l, 2l+1 of the group as a float2 (packed FFMA2 arithmetic), the per-cell vectors live once per group
// in shared memory ([species][lane] float2: 0.5 KB per species), and the species dimension of every phase is split
// over the four warps -- a quarter of the shared memory per warp (12 warps per SM) and a quarter of the serial work
// per thread:
//   phase 1  x_k = Y_k/W_k, thermo, r_k = 1/ghat_k, conductivity   species k = w, w+4, ...; partial sums combined
//            through shared memory.  (x_k is never normalised to X_k: Wilke's ratio does not care, the conductivity
//            and S_k are corrected by sum(x) at the end -- so nothing here waits for a sum over species)
//   phase 3  Wilke: warp w owns rows k in [w Kp/4, (w+1) Kp/4) (accumulators in registers) and streams all j:
//            den_k += B_kj (X_j + g_k (2 X_j r_j + g_k X_j r_j^2)) -- three FFMA2 per (k, j), B_kj from a table re-tiled
//            per warp so that a row segment is four broadcast LDS.128.  When the mechanism's weights allow it (mech.cu) B is
//            held factored, B = U diag(s) V^T cut after 8 or 12 terms: warp w projects the three vectors on the modes w, w + 4,
//            w + 8, one barrier, then expands its rows -- 6 r K FMAs instead of 3 K^2
//   phase 4  mixture-averaged diffusion: the Kp species form EIGHT tiles of TS = Kp/8, each symmetric pair of species is
//            evaluated once (4 FFMA2 Horner, two MUFU.RCP, 2 FFMA2).  The 28 off-diagonal tile pairs are played as a
//            round-robin tournament of 8 teams: 7 rounds x 4 pairs with pairwise disjoint tiles, one pair per warp, so
//            the four warps add into the shared S accumulators without atomics and every round is balanced; two more
//            rounds take the 8 diagonal tiles.  One block barrier per round.  A warp stages its own coefficient tile
//            (<= 1280 B, in loop order) with cp.async one round ahead.
//   final    D_k = N_k / S_k, N_k = sum_{j != k} Y_j evaluated as (sum_j Y_j) - Y_k with the sum formed in fp64 over the
//            exact fp32 Y (phase 1, where Y is converted for the enthalpy anyway) and handed on as an unevaluated
//            float-float pair: what A7 warns of is the rounding of the fp32 sum, amplified by the cancellation; the
//            pair is exact to ~1e-14 sum Y.  Self-diffusion D_kk when S_k = 0.
// A block is one group; it loops over groups (grid-stride) so the tables are staged once per block.
#include "common.cuh"

namespace {

constexpr int kGT = 128;       // threads per block = 4 warps sharing 64 cells
constexpr int kGroupCells = 64;
typedef float2 f2;
__device__ __forceinline__ f2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 fma2(f2 a, float s, f2 c) { return __ffma2_rn(a, bc(s), c); }
__device__ __forceinline__ f2 fma2(f2 a, float s, float c) { return __ffma2_rn(a, bc(s), bc(c)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 mul2(f2 a, float s) { return __fmul2_rn(a, bc(s)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
// one MUFU.RCP per half (B200's XU pipe is far from full here: the shared form 1/x = y/(xy), one MUFU + three FMUL, on any
// share of the pairs measured 0-1.5 % slower)
__device__ __forceinline__ f2 rcp2(f2 a) { return make_float2(rcp_approx(a.x), rcp_approx(a.y)); }
// hi + lo += y with the rounding error of the addition kept (Knuth's TwoSum, packed for two cells)
__device__ __forceinline__ void two_sum_acc(f2& hi, f2& lo, f2 y) {
    const f2 s = add2(hi, y);
    const f2 bb = add2(s, make_float2(-hi.x, -hi.y));
    const f2 e = add2(add2(hi, make_float2(bb.x - s.x, bb.y - s.y)), add2(y, make_float2(-bb.x, -bb.y)));
    hi = s;
    lo = add2(lo, e);
}
__device__ __forceinline__ f2 poly4_2(float c0, float c1, float c2, float c3, float c4, f2 u) {
    return fma2(fma2(fma2(fma2(u, c4, c3), u, bc(c2)), u, bc(c1)), u, bc(c0));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int kTileFloatsMax = 8 * 40;   // ring slot: the largest tile (TS = 8: 8 rows of 8 pairs x 5 coefficients)
__host__ __device__ constexpr int tile_row_floats(int TS) { return (TS * 5 + 3) / 4 * 4; }   // rows start 16-byte aligned

// round-robin tournament of the 8 species tiles (circle method), then the diagonal tiles: [round][warp], one word per
// entry: kt | jt << 4 | tile << 8, tile = kt * 8 - kt (kt - 1) / 2 + (jt - kt) the index of the (kt <= jt) tile in the table
#define DF_T(kt, jt) ((kt) | ((jt) << 4) | (((kt) * 8 - (kt) * ((kt) - 1) / 2 + ((jt) - (kt))) << 8))
__constant__ int kSched[9][4] = {
    {DF_T(0, 7), DF_T(1, 6), DF_T(2, 5), DF_T(3, 4)}, {DF_T(0, 6), DF_T(5, 7), DF_T(1, 4), DF_T(2, 3)},
    {DF_T(0, 5), DF_T(4, 6), DF_T(3, 7), DF_T(1, 2)}, {DF_T(0, 4), DF_T(3, 5), DF_T(2, 6), DF_T(1, 7)},
    {DF_T(0, 3), DF_T(2, 4), DF_T(1, 5), DF_T(6, 7)}, {DF_T(0, 2), DF_T(1, 3), DF_T(4, 7), DF_T(5, 6)},
    {DF_T(0, 1), DF_T(2, 7), DF_T(3, 6), DF_T(4, 5)}, {DF_T(0, 0), DF_T(1, 1), DF_T(2, 2), DF_T(3, 3)},
    {DF_T(4, 4), DF_T(5, 5), DF_T(6, 6), DF_T(7, 7)}};
#undef DF_T
constexpr int kRounds = 9;

// One TS x TS tile of species pairs.  coef: [a][b][5] in shared memory (warp-uniform addresses: broadcast loads).
// NB: columns b < NB of the j tile are evaluated -- TS, or the first half when the rest of the last tile is padding.
template <int TS, bool DIAG, int NB>
__device__ __forceinline__ void diff_tile(const float* __restrict__ coef, f2 u, const f2 (&Xk)[TS], const f2 (&Xj)[TS],
                                          f2 (&Sk)[TS], f2 (&Sj)[TS]) {
    constexpr int RS = tile_row_floats(TS), NQ = (5 * NB + 3) / 4;
#pragma unroll
    for (int a = 0; a < (DIAG ? TS - 1 : TS); ++a) {
        float q[4 * NQ];
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
            const float4 v = reinterpret_cast<const float4*>(coef + a * RS)[i];
            q[4 * i] = v.x; q[4 * i + 1] = v.y; q[4 * i + 2] = v.z; q[4 * i + 3] = v.w;
        }
#pragma unroll
        for (int b = DIAG ? a + 1 : 0; b < NB; ++b) {
            const f2 P = poly4_2(q[5 * b], q[5 * b + 1], q[5 * b + 2], q[5 * b + 3], q[5 * b + 4], u);
            const f2 r = rcp2(P);
            Sk[a] = fma2(Xj[b], r, Sk[a]);
            if (DIAG) Sk[b] = fma2(Xk[a], r, Sk[b]);
            else Sj[b] = fma2(Xk[a], r, Sj[b]);
        }
    }
}

constexpr int kScrSlots = 14;   // per warp and lane: float2-sized exchange slots (sum x, 5 C, 2 H0, s1, s2, acc, 2 sum Y)
constexpr int kSmallStride = 20;

struct GroupSmem {   // byte offsets into the dynamic shared memory of a block
    int sX, sR, small, thp, h0p, BW, ring, scr, total;
};
__host__ __device__ inline GroupSmem group_smem(int Kp, int wilke_rank) {
    GroupSmem g;
    int o = 0;
    g.sX = o; o += Kp * 32 * 8;
    g.sR = o; o += Kp * 32 * 8;
    g.h0p = o; o += Kp * 2 * 8;
    g.small = o; o += Kp * kSmallStride * 4;
    g.thp = o; o += Kp * 12 * 4;
    g.BW = o; o += wilke_rank ? (4 * Kp * 4 + 4 * wilke_rank * 16) * 4 : 4 * Kp * 16 * 4;   // factored: VW then UW
    g.ring = o; o += 4 * 2 * kTileFloatsMax * 4;   // per warp: two coefficient tiles
    g.scr = o; o += 4 * kScrSlots * 32 * 8;
    g.total = o;
    return g;
}

// KW: Wilke rows per warp = Kp / 4.  FULL: every group of the launch lies inside the field (the host launches the ragged
// last group separately), so loads and stores are plain float2 accesses.  ALL: all five outputs are wanted (the solver's
// call), so none of the per-species code is guarded by a runtime flag.
// NM: 0, or a quarter of the number of terms of Wilke's B in its factored form (MechDev::VW, UW: 2 or 3 modes per warp).
template <int KW, bool FULL, bool ALL, int NM>
__global__ void __launch_bounds__(kGT, 3)
props_group_kernel(const __grid_constant__ MechDev md, long long g_first, long long g_end, long long n, long long ld, const float* __restrict__ Tg,
                   const float* __restrict__ pg, const float* __restrict__ Yg, float* __restrict__ cp_o,
                   float* __restrict__ h_o, float* __restrict__ mu_o, float* __restrict__ lam_o, float* __restrict__ D_o) {
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int Kp = 4 * KW, TS = KW / 2;   // eight species tiles of TS
    const int K = md.K;
    constexpr bool LR = NM > 0;
    constexpr int kRank = 4 * NM;
    const GroupSmem L = group_smem(Kp, kRank);
    f2* sX = reinterpret_cast<f2*>(smem + L.sX);
    f2* sR = reinterpret_cast<f2*>(smem + L.sR);
    const double* sH0 = reinterpret_cast<const double*>(smem + L.h0p);
    const float* sSmall = reinterpret_cast<const float*>(smem + L.small);
    const float* sTh = reinterpret_cast<const float*>(smem + L.thp);
    const float* sBW = reinterpret_cast<const float*>(smem + L.BW);
    float* sRing = reinterpret_cast<float*>(smem + L.ring);
    f2* sScr = reinterpret_cast<f2*>(smem + L.scr);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;

    // ---- stage the tables once per block ----
    for (int e = tid; e < Kp * 2; e += kGT) reinterpret_cast<double*>(smem + L.h0p)[e] = md.h0p[e];
    for (int e = tid; e < Kp * kSmallStride / 4; e += kGT)
        reinterpret_cast<float4*>(smem + L.small)[e] = __ldg(reinterpret_cast<const float4*>(md.small_p) + e);
    for (int e = tid; e < Kp * 12 / 4; e += kGT)
        reinterpret_cast<float4*>(smem + L.thp)[e] = __ldg(reinterpret_cast<const float4*>(md.thp) + e);
    if (LR) {
        for (int e = tid; e < Kp * 4; e += kGT)
            reinterpret_cast<float4*>(smem + L.BW)[e] = __ldg(reinterpret_cast<const float4*>(md.VW) + e);
        for (int e = tid; e < 4 * kRank * 4; e += kGT) {   // UW[w][m < kRank][16], rows of kWilkeRank in global memory
            const int ww = e / (kRank * 4), rest = e % (kRank * 4);
            reinterpret_cast<float4*>(smem + L.BW)[Kp * 4 + e] = __ldg(reinterpret_cast<const float4*>(md.UW) + ww * kWilkeRank * 4 + rest);
        }
    } else {
        for (int e = tid; e < 4 * Kp * 16 / 4; e += kGT)
            reinterpret_cast<float4*>(smem + L.BW)[e] = __ldg(reinterpret_cast<const float4*>(md.BW) + e);
    }
    __syncthreads();

    const bool want_h = ALL || h_o, want_cp = ALL || cp_o, want_mu = ALL || mu_o, want_lam = ALL || lam_o, want_D = ALL || D_o;
    const bool want_thermo = want_cp || want_h, want_transport = want_mu || want_lam || want_D;
    const long long ngroups = g_end;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(sRing + w * 2 * kTileFloatsMax);   // this warp's two coefficient slots
    // T and p of a group are loaded one group ahead (their latency would otherwise open every group)
    auto ld2_at = [&](const float* p, long long grp) -> f2 {
        const long long ir = grp * kGroupCells + 2 * lane;
        if (FULL || ir + 1 < n) return __ldg(reinterpret_cast<const float2*>(p + ir));
        const float v = __ldg(p + (ir < n ? ir : 0));
        return make_float2(v, v);
    };
    f2 T_next = bc(1000.f), p_next = bc(1.f);
    if (g_first + blockIdx.x < ngroups) {
        T_next = ld2_at(Tg, g_first + blockIdx.x);
        if (want_D) p_next = ld2_at(pg, g_first + blockIdx.x);
    }
    for (long long grp = g_first + blockIdx.x; grp < ngroups; grp += gridDim.x) {
        // every thread stays alive through the barriers; lanes past the end of the field work on cell 0 and do not store
        const long long i_raw = grp * kGroupCells + 2 * lane;
        const bool valid = FULL || i_raw < n;
        const long long i = valid ? i_raw : 0;
        const bool two = FULL || (valid && (i + 1 < n));
        auto ld2 = [&](const float* p) -> f2 {
            if (two) return __ldg(reinterpret_cast<const float2*>(p + i));
            const float v = __ldg(p + i);
            return make_float2(v, v);
        };
        auto st2 = [&](float* p, f2 v) {
            if (two) *reinterpret_cast<float2*>(p + i) = v;
            else if (valid) p[i] = v.x;
        };
        const f2 T = T_next, p_cell = p_next;
        // all of this warp's Y rows in flight at once, then the next group's T and p
        f2 yv[KW];
#pragma unroll
        for (int a = 0; a < KW; ++a) yv[a] = (a < KW - 2 || w + 4 * a < K) ? ld2(Yg + (size_t)(w + 4 * a) * ld) : bc(0.f);   // K > Kp - 8
        if (grp + gridDim.x < ngroups) {
            T_next = ld2_at(Tg, grp + gridDim.x);
            if (want_D) p_next = ld2_at(pg, grp + gridDim.x);
        }
        const f2 tau = mul2(add2(T, bc(-md.sc.T_mid)), md.sc.inv_S);
        const bool lo0 = T.x < md.sc.T_mid, lo1 = T.y < md.sc.T_mid;   // A2: hi for T >= T_mid
        const f2 u = mul2(add2(make_float2(logf(T.x), logf(T.y)), bc(-md.sc.Lc)), md.sc.inv_Ls);
        const f2 sqrtT = make_float2(sqrtf(T.x), sqrtf(T.y));

        // ---- phase 1: x_k = Y_k / W_k and the thermo sums of this warp's species --------------------------------
        {
            // both ranges are accumulated and the range is picked after the exchange: ten FFMA2 per species instead of
            // five FFMA2 + ten selects (the exchange grows by five slots, which costs nothing)
            f2 Cl[5], Ch[5];
#pragma unroll
            for (int m = 0; m < 5; ++m) Cl[m] = Ch[m] = bc(0.f);
            double H0la = 0.0, H0ha = 0.0, H0lb = 0.0, H0hb = 0.0, Yta = 0.0, Ytb = 0.0;
            f2 sumx = bc(0.f), s1 = bc(0.f), s2 = bc(0.f);
#pragma unroll
            for (int a = 0; a < KW; ++a) {
                const int k = w + 4 * a;
                const f2 y = yv[a];
                const float4 ta = *reinterpret_cast<const float4*>(sSmall + k * kSmallStride);   // invW sqrtW v0 v1
                const f2 x = mul2(y, ta.x);
                sX[k * 32 + lane] = x;
                sumx = add2(sumx, x);
                if (want_transport) {   // r_k = 1/ghat_k and the conductivity sums, on the unnormalised x_k
                    const float4 tb = *reinterpret_cast<const float4*>(sSmall + k * kSmallStride + 4),   // v2 v3 v4 c0
                                 tc = *reinterpret_cast<const float4*>(sSmall + k * kSmallStride + 8);   // c1 c2 c3 c4
                    sR[k * 32 + lane] = rcp2(poly4_2(ta.z, ta.w, tb.x, tb.y, tb.z, u));
                    const f2 lk = poly4_2(tb.w, tc.x, tc.y, tc.z, tc.w, u);
                    s1 = fma2(x, lk, s1);
                    s2 = fma2(x, rcp2(lk), s2);
                }
                if (want_h || want_D) {
                    const double ya = (double)y.x, yb = (double)y.y;
                    if (want_D) {   // sum_j Y_j in fp64 (exact on the fp32 inputs to 1e-16): N_k = sum - Y_k without the fp32 rounding of the sum
                        Yta += ya;
                        Ytb += yb;
                    }
                    if (want_h) {   // formation-enthalpy term in fp64 (|h| ~ 1e7 J/kg against a 1e-5 tolerance)
                        const double hl = sH0[2 * k], hh = sH0[2 * k + 1];
                        H0la = fma(ya, hl, H0la); H0ha = fma(ya, hh, H0ha);
                        H0lb = fma(yb, hl, H0lb); H0hb = fma(yb, hh, H0hb);
                    }
                }
                if (want_thermo) {
                    const float4 a4 = *reinterpret_cast<const float4*>(sTh + k * 12), b4 = *reinterpret_cast<const float4*>(sTh + k * 12 + 4),
                                 c4 = *reinterpret_cast<const float4*>(sTh + k * 12 + 8);   // lo c0..c5 | hi c0..c5
                    Cl[0] = fma2(y, a4.y, Cl[0]); Cl[1] = fma2(y, a4.z, Cl[1]); Cl[2] = fma2(y, a4.w, Cl[2]);
                    Cl[3] = fma2(y, b4.x, Cl[3]); Cl[4] = fma2(y, b4.y, Cl[4]);
                    Ch[0] = fma2(y, b4.w, Ch[0]); Ch[1] = fma2(y, c4.x, Ch[1]); Ch[2] = fma2(y, c4.y, Ch[2]);
                    Ch[3] = fma2(y, c4.z, Ch[3]); Ch[4] = fma2(y, c4.w, Ch[4]);
                }
            }
            f2* my = sScr + (w * kScrSlots) * 32 + lane;
            my[0] = sumx;
            my[8 * 32] = s1;
            my[9 * 32] = s2;
            if (want_D) {   // the warp's share of sum Y as a float-float pair
                const f2 hi = make_float2((float)Yta, (float)Ytb);
                my[11 * 32] = hi;
                my[12 * 32] = make_float2((float)(Yta - (double)hi.x), (float)(Ytb - (double)hi.y));
            }
            if (want_thermo) {
#pragma unroll
                for (int m = 0; m < 5; ++m) my[(1 + m) * 32] = make_float2(lo0 ? Cl[m].x : Ch[m].x, lo1 ? Cl[m].y : Ch[m].y);
                reinterpret_cast<double*>(my)[6 * 32] = lo0 ? H0la : H0ha;
                reinterpret_cast<double*>(my)[7 * 32] = lo1 ? H0lb : H0hb;
            }
        }
        __syncthreads();
        f2 sumx = bc(0.f);
#pragma unroll
        for (int v = 0; v < 4; ++v) sumx = add2(sumx, sScr[(v * kScrSlots) * 32 + lane]);
        if (want_thermo && w == 1) {
            f2 q[5];
#pragma unroll
            for (int m = 0; m < 5; ++m) {
                q[m] = bc(0.f);
#pragma unroll
                for (int v = 0; v < 4; ++v) q[m] = add2(q[m], sScr[(v * kScrSlots + 1 + m) * 32 + lane]);
            }
            if (want_cp)
                st2(cp_o, mul2(fma2(fma2(fma2(fma2(mul2(q[4], 5.f), tau, mul2(q[3], 4.f)), tau, mul2(q[2], 3.f)), tau,
                                         mul2(q[1], 2.f)), tau, q[0]),
                               md.sc.inv_S));
            if (want_h) {
                double Ha = 0.0, Hb = 0.0;
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    Ha += reinterpret_cast<const double*>(sScr + (v * kScrSlots) * 32 + lane)[6 * 32];
                    Hb += reinterpret_cast<const double*>(sScr + (v * kScrSlots) * 32 + lane)[7 * 32];
                }
                const f2 sens = mul2(tau, fma2(fma2(fma2(fma2(q[4], tau, q[3]), tau, q[2]), tau, q[1]), tau, q[0]));
                st2(h_o, make_float2((float)(Ha + (double)sens.x), (float)(Hb + (double)sens.y)));
            }
        }
        if (!want_transport) {   // block-uniform
            __syncthreads();     // the scratch is rewritten by the next group
            continue;
        }

        // Mole fractions are never normalised: with x_k = Y_k/W_k = X_k sum(x), Wilke's ratio is unchanged (numerator and
        // denominator both carry sum(x)), and the conductivity sums and S_k are corrected by sum(x) where they are used.
        // That makes phase 2 (r_k, conductivity) independent of any sum over species: it runs inside phase 1's loop.
        if (want_lam && w == 0) {
            f2 s1 = bc(0.f), s2 = bc(0.f);
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                s1 = add2(s1, sScr[(v * kScrSlots + 8) * 32 + lane]);
                s2 = add2(s2, sScr[(v * kScrSlots + 9) * 32 + lane]);
            }
            // A6 with X = x / sum(x): sum X lk = s1 / sum(x), 1 / sum(X / lk) = sum(x) / s2
            st2(lam_o, mul2(mul2(sqrtT, 0.5f), add2(mul2(s1, rcp2(sumx)), mul2(sumx, rcp2(s2)))));
        }

        // ---- phase 3: Wilke; this warp owns rows k0 .. k0 + KW - 1 ------------------------------------------------
        if (want_mu) {
            const int k0 = w * KW;
            f2 gk[KW], den[KW];
#pragma unroll
            for (int a = 0; a < KW; ++a) {
                gk[a] = rcp2(sR[(k0 + a) * 32 + lane]);
                den[a] = bc(0.f);
            }
            if constexpr (LR) {
                // den_k = sum_j B_kj (x_j + 2 g_k x_j r_j + g_k^2 x_j r_j^2) with B = U diag(s) V^T cut after kRank terms
                // (kRank = 8 or 12 terms, 1e-6; B is a smooth function of W_k/W_j): first the three vectors projected on the V_m -- warp w takes the
                // modes w, w + 4, w + 8 over all species --, then, after a barrier, the rows of this warp from the U_m:
                // 6 r K packed FMAs per group instead of 3 K^2.
                f2 tP[NM], tQ[NM], tR[NM];
#pragma unroll
                for (int c = 0; c < NM; ++c) tP[c] = tQ[c] = tR[c] = bc(0.f);
                const float4* vw = reinterpret_cast<const float4*>(sBW) + (size_t)w * Kp;
#pragma unroll 4
                for (int j = 0; j < K; ++j) {
                    const f2 xj = sX[j * 32 + lane], rj = sR[j * 32 + lane];
                    const f2 xr = mul2(xj, rj), xrr = mul2(xr, rj);
                    const float4 v = vw[j];
                    const float vm[3] = {v.x, v.y, v.z};   // modes w, w + 4, w + 8
#pragma unroll
                    for (int c = 0; c < NM; ++c) {
                        tP[c] = fma2(xj, vm[c], tP[c]);
                        tQ[c] = fma2(xr, vm[c], tQ[c]);
                        tR[c] = fma2(xrr, vm[c], tR[c]);
                    }
                }
                f2* sT = reinterpret_cast<f2*>(sRing);   // [mode][3][lane]: the ring is idle until the pair rounds
#pragma unroll
                for (int c = 0; c < NM; ++c) {
                    const int m = w + 4 * c;
                    sT[(3 * m) * 32 + lane] = tP[c];
                    sT[(3 * m + 1) * 32 + lane] = add2(tQ[c], tQ[c]);
                    sT[(3 * m + 2) * 32 + lane] = tR[c];
                }
                __syncthreads();
                const float* uw = sBW + (size_t)4 * Kp * 4 + (size_t)w * kRank * 16;
#pragma unroll 2
                for (int m = 0; m < kRank; ++m) {
                    const f2 p0 = sT[(3 * m) * 32 + lane], q2 = sT[(3 * m + 1) * 32 + lane], r2 = sT[(3 * m + 2) * 32 + lane];
                    float U[16];
#pragma unroll
                    for (int q4 = 0; q4 < (KW + 3) / 4; ++q4) {
                        const float4 v = *reinterpret_cast<const float4*>(uw + m * 16 + 4 * q4);
                        U[4 * q4] = v.x; U[4 * q4 + 1] = v.y; U[4 * q4 + 2] = v.z; U[4 * q4 + 3] = v.w;
                    }
#pragma unroll
                    for (int a = 0; a < KW; ++a) den[a] = fma2(fma2(gk[a], fma2(gk[a], r2, q2), p0), U[a], den[a]);
                }
            }
            const float* bw = sBW + (size_t)w * Kp * 16;
#pragma unroll 2
            for (int j = 0; j < (LR ? 0 : K); ++j) {   // padding species have X_j = 0: skipped
                const f2 xj = sX[j * 32 + lane], rj = sR[j * 32 + lane];
                const f2 xr = mul2(xj, rj);
                const f2 b2 = add2(xr, xr), c = mul2(xr, rj);
                float B[16];
#pragma unroll
                for (int q4 = 0; q4 < (KW + 3) / 4; ++q4) {
                    const float4 v = *reinterpret_cast<const float4*>(bw + j * 16 + 4 * q4);
                    B[4 * q4] = v.x; B[4 * q4 + 1] = v.y; B[4 * q4 + 2] = v.z; B[4 * q4 + 3] = v.w;
                }
#pragma unroll
                for (int a = 0; a < KW; ++a)   // B_kj X_j (1 + g_k r_j)^2, expanded: all terms positive
                    den[a] = fma2(fma2(gk[a], fma2(gk[a], c, b2), xj), B[a], den[a]);
            }
            f2 acc = bc(0.f);
#pragma unroll
            for (int a = 0; a < KW; ++a)
                acc = fma2(mul2(mul2(sX[(k0 + a) * 32 + lane], sSmall[(k0 + a) * kSmallStride + 1]), mul2(gk[a], gk[a])), rcp2(den[a]), acc);
            sScr[(w * kScrSlots + 10) * 32 + lane] = acc;
        }
        __syncthreads();   // every warp is done reading r: sR becomes the S accumulators
        if (want_mu && w == 0) {
            f2 acc = bc(0.f);
#pragma unroll
            for (int v = 0; v < 4; ++v) acc = add2(acc, sScr[(v * kScrSlots + 10) * 32 + lane]);
            st2(mu_o, mul2(sqrtT, acc));
        }
        if (!want_D) continue;   // block-uniform; the barrier above also protects the scratch

        // ---- phase 4: mixture-averaged diffusivities ---------------------------------------------------------------
        for (int k = w; k < Kp; k += 4) sR[k * 32 + lane] = bc(0.f);
        // the next group's Y rows on their way from HBM to L2 while this group's pair loops run
        if (grp + gridDim.x < ngroups && (lane & 7) == 0) {
            const long long in = (grp + gridDim.x) * kGroupCells + 2 * lane;
            if (in < n) {
#pragma unroll
                for (int a = 0; a < KW; ++a)
                    if (a < KW - 2 || w + 4 * a < K) asm volatile("prefetch.global.L2 [%0];" ::"l"(Yg + (size_t)(w + 4 * a) * ld + in));
            }
        }
        constexpr int kTileFloats = TS * tile_row_floats(TS), kTile16 = kTileFloats / 4;
        const float* ring = sRing + w * 2 * kTileFloatsMax;
        auto stage = [&](int sched, int buf) {   // the whole tile is one or two 16-byte pieces per lane
            const float* src = md.dtile + (size_t)(sched >> 8) * kTileFloats + 4 * lane;
            const uint32_t dst = ring_s + (buf * kTileFloatsMax + 4 * lane) * 4;
#pragma unroll
            for (int c = 0; c < (kTile16 + 31) / 32; ++c)
                if ((c + 1) * 32 <= kTile16 || lane + c * 32 < kTile16)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + c * 512), "l"(src + c * 128) : "memory");
            cp_async_commit();
        };
        int sched = kSched[0][w];
        stage(sched, 0);
        __syncthreads();   // S is zeroed everywhere
        for (int r = 0; r < kRounds; ++r) {
            const int sched_next = kSched[r + 1 < kRounds ? r + 1 : r][w];
            if (r + 1 < kRounds) stage(sched_next, (r + 1) & 1);
            else cp_async_commit();
            cp_async_wait<1>();
            __syncwarp();
            const int kt = sched & 15, jt = (sched >> 4) & 15;
            sched = sched_next;
            const float* coef = ring + (r & 1) * kTileFloatsMax;
            f2 Xk[TS], Xj[TS], Sk[TS], Sj[TS];
            const f2* xk = sX + kt * TS * 32 + lane;
            const f2* xj = sX + jt * TS * 32 + lane;
#pragma unroll
            for (int a = 0; a < TS; ++a) {
                Xk[a] = xk[a * 32];
                Xj[a] = xj[a * 32];
                Sk[a] = Sj[a] = bc(0.f);
            }
            // block-uniform: the two diagonal rounds.  Warp-uniform: the tile whose j side is the last species tile, when at
            // least half of that tile is padding (K = 53: species 53..55 of 49..55), evaluates the first half only -- that warp
            // waits at the round's barrier either way, but the SM's other blocks get its issue slots
            constexpr int NBH = (TS + 1) / 2;
            if (r >= 7) diff_tile<TS, true, TS>(coef, u, Xk, Xj, Sk, Sj);
            else if (jt == 7 && K - 7 * TS <= NBH) diff_tile<TS, false, NBH>(coef, u, Xk, Xj, Sk, Sj);
            else diff_tile<TS, false, TS>(coef, u, Xk, Xj, Sk, Sj);
            // tiles kt and jt of S belong to this warp alone in this round
            f2* sk = sR + kt * TS * 32 + lane;
#pragma unroll
            for (int a = 0; a < TS; ++a) sk[a * 32] = add2(sk[a * 32], Sk[a]);
            if (r < 7) {
                f2* sj = sR + jt * TS * 32 + lane;
#pragma unroll
                for (int a = 0; a < TS; ++a) sj[a * 32] = add2(sj[a * 32], Sj[a]);
            }
            __syncthreads();
        }
        cp_async_wait<0>();

        // ---- final: D_k = N_k / S_k for this warp's species k = w, w + 4, ... (its Y rows again: L2 hits) ------------
        {
#pragma unroll
            for (int a = 0; a < KW; ++a) yv[a] = (a < KW - 2 || w + 4 * a < K) ? ld2(Yg + (size_t)(w + 4 * a) * ld) : bc(0.f);
            f2 thi = bc(0.f), tlo = bc(0.f);
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                two_sum_acc(thi, tlo, sScr[(v * kScrSlots + 11) * 32 + lane]);
                tlo = add2(tlo, sScr[(v * kScrSlots + 12) * 32 + lane]);
            }
            const f2 scale = make_float2(T.x * sqrtT.x * rcp_approx(p_cell.x), T.y * sqrtT.y * rcp_approx(p_cell.y));
#pragma unroll
            for (int a = 0; a < KW; ++a) {
                const int k = w + 4 * a;
                if (a < KW - 2 || k < K) {
                    // (hi - Y_k) loses nothing that matters: an fp32 difference is exact to 2^-24 of its RESULT; what
                    // cancellation would amplify is the rounding of the sum itself, and that sits in lo
                    const f2 Nk = add2(add2(thi, make_float2(-yv[a].x, -yv[a].y)), tlo);
                    const f2 S = sR[k * 32 + lane];
                    const float* dd = sSmall + k * kSmallStride + 12;
                    const f2 dk = poly4_2(dd[0], dd[1], dd[2], dd[3], dd[4], u);
                    const f2 q = mul2(mul2(Nk, sumx), rcp2(S));   // S was accumulated on x = X sum(x)
                    const f2 Dk = make_float2(S.x > 0.f ? q.x : dk.x, S.y > 0.f ? q.y : dk.y);   // A7
                    st2(D_o + (size_t)k * ld, mul2(Dk, scale));
                }
            }
        }
        __syncthreads();   // sX / sR / scratch are rewritten by the next group
    }
}

template <int KW, bool FULL, bool ALL, int NM>
df_status launch_one(const MechDev& md, long long g_first, long long g_end, long long n, long long ld, const float* T, const float* p,
                     const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    const int smem = group_smem(4 * KW, 4 * NM).total;
    static DfPerDevice smem_attr;
    const df_status st = df_ensure_dyn_smem((const void*)props_group_kernel<KW, FULL, ALL, NM>, smem, &smem_attr);
    if (st != DF_OK) return st;
    const long long ngroups = g_end - g_first;
    const long long cap = (long long)df_device_sm_count() * 3 * 4;   // 3 resident blocks per SM, ~4 waves
    const long long blocks = ngroups < cap ? ngroups : cap;
    props_group_kernel<KW, FULL, ALL, NM><<<(unsigned)(blocks > 0 ? blocks : 1), kGT, smem, s>>>(md, g_first, g_end, n, ld, T, p, Y, cp, h, mu, lam, D);
    DF_CUDA_TRY(cudaGetLastError());
    return DF_OK;
}

// the full groups in one launch, the ragged last group (if any) in a launch of its own
template <int KW, int NM>
df_status launch_lr(const MechDev& md, long long n, long long ld, const float* T, const float* p, const float* Y, float* cp,
                    float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    const long long full_groups = n / kGroupCells, ngroups = (n + kGroupCells - 1) / kGroupCells;
    const bool all = cp && h && mu && lam && D;
    df_status st = DF_OK;
    if (full_groups > 0)
        st = all ? launch_one<KW, true, true, NM>(md, 0, full_groups, n, ld, T, p, Y, cp, h, mu, lam, D, s)
                 : launch_one<KW, true, false, NM>(md, 0, full_groups, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    if (st == DF_OK && ngroups > full_groups)
        st = launch_one<KW, false, false, NM>(md, full_groups, ngroups, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    return st;
}

template <int KW>
df_status launch_kw(const MechDev& md, long long n, long long ld, const float* T, const float* p, const float* Y, float* cp,
                    float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    if constexpr (KW >= 8) {   // K > 28: the factored Wilke pays when the mechanism's B allows it (mech.cu)
        if (md.wilke_rank == 8) return launch_lr<KW, 2>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        if (md.wilke_rank == 12) return launch_lr<KW, 3>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    }
    return launch_lr<KW, 0>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
}

}  // namespace

df_status launch_properties_group(const df_mech* mech, long long n, long long ld, const float* T, const float* p,
                                  const float* Y, float* cp, float* h, float* mu, float* lam, float* D, cudaStream_t s) {
    const MechDev& md = mech->dev;
    switch (md.Kp / 8) {
        case 1: return launch_kw<2>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 2: return launch_kw<4>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 3: return launch_kw<6>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 4: return launch_kw<8>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 5: return launch_kw<10>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 6: return launch_kw<12>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 7: return launch_kw<14>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
        case 8: return launch_kw<16>(md, n, ld, T, p, Y, cp, h, mu, lam, D, s);
    }
    return df_set_error(DF_ERR_UNSUPPORTED, "df_thermo_properties: K = %d", md.K);
}

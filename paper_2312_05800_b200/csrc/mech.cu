// mech.cu -- df_mech: create-time repacking of the species tables (host, fp64/long double) into
// the forms the kernels evaluate in fp32 without losing the 1e-5 / 1e-3 K tolerances:
//   * NASA-7 enthalpy polynomials re-expanded about T_mid in tau = (T - T_mid)/S   (K1)
//   * ln T fits re-expanded in u = (ln T - Lc)/Ls, |u| <~ 1                        (K2)
//   * Wilke's mass-ratio factor tabulated as B_kj and W_k^(-1/4) folded into the viscosity fit.
#include <cmath>
#include <cstring>
#include <new>
#include <utility>

#include "common.cuh"

namespace {

// q(x) = p(c + s x): coefficients of the shifted/scaled polynomial, degree n-1.
void shift_poly(const long double* p, int n, long double c, long double s, long double* q) {
    for (int m = 0; m < n; ++m) {
        long double acc = 0.0L, binom = 1.0L, cpow = 1.0L;  // C(i,m) c^(i-m), i = m..n-1
        for (int i = m; i < n; ++i) {
            acc += p[i] * binom * cpow;
            binom = binom * (long double)(i + 1) / (long double)(i + 1 - m);
            cpow *= c;
        }
        q[m] = acc * powl(s, m);
    }
}

// One-sided Jacobi SVD (Hestenes) of a K x K matrix in fp64: A = U diag(s) V^T, s descending.  A is overwritten by U diag(s).
void jacobi_svd(int K, std::vector<double>& A, std::vector<double>& V, std::vector<double>& s) {
    V.assign((size_t)K * K, 0.0);
    for (int i = 0; i < K; ++i) V[(size_t)i * K + i] = 1.0;
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0.0;
        for (int p = 0; p < K - 1; ++p)
            for (int q = p + 1; q < K; ++q) {
                double a = 0.0, b = 0.0, c = 0.0;
                for (int i = 0; i < K; ++i) {
                    const double x = A[(size_t)i * K + p], y = A[(size_t)i * K + q];
                    a += x * x; b += y * y; c += x * y;
                }
                if (fabs(c) <= 1e-300) continue;
                off = fmax(off, fabs(c) / sqrt(fmax(a * b, 1e-300)));
                const double zeta = (b - a) / (2.0 * c);
                const double tq = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                const double cs = 1.0 / sqrt(1.0 + tq * tq), sn = cs * tq;
                for (int i = 0; i < K; ++i) {
                    double x = A[(size_t)i * K + p], y = A[(size_t)i * K + q];
                    A[(size_t)i * K + p] = cs * x - sn * y;
                    A[(size_t)i * K + q] = sn * x + cs * y;
                    x = V[(size_t)i * K + p]; y = V[(size_t)i * K + q];
                    V[(size_t)i * K + p] = cs * x - sn * y;
                    V[(size_t)i * K + q] = sn * x + cs * y;
                }
            }
        if (off < 1e-15) break;
    }
    s.assign(K, 0.0);   // column norms = singular values; then sort descending
    for (int j = 0; j < K; ++j) {
        double n2 = 0.0;
        for (int i = 0; i < K; ++i) n2 += A[(size_t)i * K + j] * A[(size_t)i * K + j];
        s[j] = sqrt(n2);
    }
    for (int j = 0; j < K; ++j) {
        int best = j;
        for (int l = j + 1; l < K; ++l)
            if (s[l] > s[best]) best = l;
        if (best != j) {
            std::swap(s[j], s[best]);
            for (int i = 0; i < K; ++i) {
                std::swap(A[(size_t)i * K + j], A[(size_t)i * K + best]);
                std::swap(V[(size_t)i * K + j], V[(size_t)i * K + best]);
            }
        }
    }
}

template <typename T>
df_status to_device(T** dst, const std::vector<T>& src) {
    *dst = nullptr;
    if (src.empty()) return DF_OK;
    DF_CUDA_TRY(cudaMalloc((void**)dst, src.size() * sizeof(T)));
    DF_CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return DF_OK;
}

struct HostTables {
    int K;
    MechScalars sc;
    std::vector<float> th32, sth32, invW, sqrtW, visc, cond, ddiag, dfull, wilkeB;
    std::vector<double> th64;
};

template <int K>
PropTables<K>* make_fixed(const HostTables& t, const double* W) {
    PropTables<K>* p = new PropTables<K>;
    memset(p, 0, sizeof(*p));
    for (int k = 0; k < K; ++k) {
        for (int r = 0; r < 2; ++r) {
            p->h0[k][r] = t.th64[(k * 2 + r) * 6];
            for (int m = 1; m < 6; ++m) p->th[k][r][m - 1] = t.th32[(k * 2 + r) * 6 + m];
        }
        p->invW[k] = t.invW[k];
        p->sqrtW[k] = t.sqrtW[k];
        for (int m = 0; m < 5; ++m) {
            p->visc[k][m] = t.visc[k * 5 + m];
            p->cond[k][m] = t.cond[k * 5 + m];
            p->ddiag[k][m] = t.ddiag[k * 5 + m];
        }
        for (int j = 0; j < K; ++j) p->B[k][j] = t.wilkeB[k * K + j];
    }
    int idx = 0;
    for (int j = 0; j < K; ++j)
        for (int k = j + 1; k < K; ++k, ++idx)
            for (int m = 0; m < 5; ++m) p->dpair[idx][m] = t.dfull[(j * K + k) * 5 + m];
    p->sc = t.sc;
    // factored Wilke (see MechDev::wilke_rank): the smallest of 7, 8 terms that reproduces every B_kj to 1e-6, if it is
    // cheaper than the K x K table (2 r < K)
    if (K > 16) {
        std::vector<double> A((size_t)K * K), Bd((size_t)K * K), V, sv;
        for (int k = 0; k < K; ++k)
            for (int j = 0; j < K; ++j) Bd[(size_t)k * K + j] = 1.0 / sqrt(8.0 * (1.0 + W[k] / W[j]));
        A = Bd;
        jacobi_svd(K, A, V, sv);
        for (int r = 7; r <= 8 && !p->wilke_rank; ++r) {
            double worst = 0.0;
            for (int k = 0; k < K; ++k)
                for (int j = 0; j < K; ++j) {
                    double acc = 0.0;
                    for (int m = 0; m < r; ++m) acc += A[(size_t)k * K + m] * V[(size_t)j * K + m];
                    worst = fmax(worst, fabs(acc / Bd[(size_t)k * K + j] - 1.0));
                }
            if (worst <= 1e-6) p->wilke_rank = r;
        }
        for (int k = 0; k < K; ++k)
            for (int m = 0; m < p->wilke_rank; ++m) {
                p->WU[k][m] = (float)A[(size_t)k * K + m];
                p->WV[k][m] = (float)V[(size_t)k * K + m];
            }
    }
    return p;
}

}  // namespace

extern "C" df_status df_mech_create(df_mech** out, int K, const double* W, const double* nasa_lo,
                                    const double* nasa_hi, double T_low, double T_mid, double T_high,
                                    const double* visc_fit, const double* cond_fit, const double* bdiff_fit) {
    if (!out) return df_set_error(DF_ERR_INVALID_ARG, "df_mech_create: out is NULL");
    *out = nullptr;
    if (!W || !nasa_lo || !nasa_hi || !visc_fit || !cond_fit || !bdiff_fit)
        return df_set_error(DF_ERR_INVALID_ARG, "df_mech_create: NULL table");
    if (K < 1 || K > DF_MAX_K) return df_set_error(DF_ERR_UNSUPPORTED, "df_mech_create: K=%d outside [1,%d]", K, DF_MAX_K);
    if (!(T_low > 0.0) || !(T_mid > T_low) || !(T_high > T_mid))
        return df_set_error(DF_ERR_INVALID_ARG, "df_mech_create: need 0 < T_low < T_mid < T_high");
    for (int k = 0; k < K; ++k)
        if (!(W[k] > 0.0)) return df_set_error(DF_ERR_INVALID_ARG, "df_mech_create: W[%d] <= 0", k);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return df_set_error(DF_ERR_CUDA, "df_mech_create: no CUDA device (there is no CPU fallback)");

    HostTables t;
    t.K = K;
    const long double S = 1000.0L;
    t.sc.T_mid = (float)T_mid;
    t.sc.S = (float)S;
    t.sc.inv_S = (float)(1.0L / S);
    t.sc.tau_min = (float)((50.0L - T_mid) / S);
    t.sc.tau_max = (float)((6000.0L - T_mid) / S);
    const long double lnlo = logl((long double)T_low), lnhi = logl((long double)T_high);
    const long double Lc = 0.5L * (lnlo + lnhi), Ls = 0.55L * (lnhi - lnlo);
    t.sc.Lc = (float)Lc;
    t.sc.inv_Ls = (float)(1.0L / Ls);
    // The kernels compute u = (ln T - (float)Lc) * (float)(1/Ls); re-expand about exactly those fp32 values.
    const long double Lc_f = (long double)t.sc.Lc, Ls_f = 1.0L / (long double)t.sc.inv_Ls;
    const long double S_f = 1.0L / (long double)t.sc.inv_S, Tm_f = (long double)t.sc.T_mid;

    t.th32.resize((size_t)K * 12);
    t.th64.resize((size_t)K * 12);
    t.sth32.resize((size_t)K * 12);
    t.invW.resize(K);
    t.sqrtW.resize(K);
    t.visc.resize((size_t)K * 5);
    t.cond.resize((size_t)K * 5);
    t.ddiag.resize((size_t)K * 5);
    t.dfull.resize((size_t)K * K * 5);
    t.wilkeB.resize((size_t)K * K);
    for (int k = 0; k < K; ++k) {
        const long double RW = (long double)DF_R_UNIVERSAL / (long double)W[k];
        for (int r = 0; r < 2; ++r) {
            const double* a = (r == 0 ? nasa_lo : nasa_hi) + 7 * k;
            // h_k/W_k = RW (a6 + a1 T + a2 T^2/2 + a3 T^3/3 + a4 T^4/4 + a5 T^5/5)
            long double p[6] = {(long double)a[5], (long double)a[0], (long double)a[1] / 2, (long double)a[2] / 3,
                                (long double)a[3] / 4, (long double)a[4] / 5};
            long double q[6];
            shift_poly(p, 6, Tm_f, S_f, q);
            for (int m = 0; m < 6; ++m) {
                t.th64[(k * 2 + r) * 6 + m] = (double)(RW * q[m]);
                t.th32[(k * 2 + r) * 6 + m] = (float)(RW * q[m]);
            }
            // s_k/W_k = RW (a1 ln T + a7 + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4): the polynomial part in tau
            long double ps[5] = {(long double)a[6], (long double)a[1], (long double)a[2] / 2, (long double)a[3] / 3,
                                 (long double)a[4] / 4};
            long double qs[5];
            shift_poly(ps, 5, Tm_f, S_f, qs);
            t.sth32[(k * 2 + r) * 6] = (float)(RW * (long double)a[0]);
            for (int m = 0; m < 5; ++m) t.sth32[(k * 2 + r) * 6 + 1 + m] = (float)(RW * qs[m]);
        }
        t.invW[k] = (float)(1.0L / (long double)W[k]);
        t.sqrtW[k] = (float)sqrtl((long double)W[k]);
        long double p[5], q[5];
        const long double w4 = powl((long double)W[k], -0.25L);
        for (int m = 0; m < 5; ++m) p[m] = (long double)visc_fit[5 * k + m];
        shift_poly(p, 5, Lc_f, Ls_f, q);
        for (int m = 0; m < 5; ++m) t.visc[k * 5 + m] = (float)(q[m] * w4);
        for (int m = 0; m < 5; ++m) p[m] = (long double)cond_fit[5 * k + m];
        shift_poly(p, 5, Lc_f, Ls_f, q);
        for (int m = 0; m < 5; ++m) t.cond[k * 5 + m] = (float)q[m];
        for (int j = 0; j < K; ++j) {
            // bdiff is declared symmetric; average the two halves so the GPU tables are exactly symmetric.
            for (int m = 0; m < 5; ++m)
                p[m] = 0.5L * ((long double)bdiff_fit[5 * ((size_t)j * K + k) + m] +
                               (long double)bdiff_fit[5 * ((size_t)k * K + j) + m]);
            shift_poly(p, 5, Lc_f, Ls_f, q);
            for (int m = 0; m < 5; ++m) t.dfull[((size_t)j * K + k) * 5 + m] = (float)q[m];
            if (j == k)
                for (int m = 0; m < 5; ++m) t.ddiag[k * 5 + m] = (float)q[m];
            t.wilkeB[(size_t)k * K + j] = (float)(1.0L / sqrtl(8.0L * (1.0L + (long double)W[k] / (long double)W[j])));
        }
    }

    df_mech* mech = new (std::nothrow) df_mech;
    if (!mech) return df_set_error(DF_ERR_ALLOC, "df_mech_create: out of host memory");
    mech->K = K;
    mech->W_host.assign(W, W + K);
    mech->th64_host = t.th64;
    MechDev& d = mech->dev;
    memset(&d, 0, sizeof(d));
    d.K = K;
    d.sc = t.sc;
    df_status st;
    if ((st = to_device(&d.th32, t.th32)) || (st = to_device(&d.sth32, t.sth32)) || (st = to_device(&d.th64, t.th64)) || (st = to_device(&d.invW, t.invW)) ||
        (st = to_device(&d.sqrtW, t.sqrtW)) || (st = to_device(&d.visc, t.visc)) || (st = to_device(&d.cond, t.cond)) ||
        (st = to_device(&d.ddiag, t.ddiag)) || (st = to_device(&d.dfull, t.dfull)) ||
        (st = to_device(&d.wilkeB, t.wilkeB))) {
        df_mech_destroy(mech);
        return st;
    }
    {   // padded / tiled tables of the any-K kernel (properties_group.cu)
        const int Kp = (K + 7) / 8 * 8, KW = Kp / 4, TS = Kp / 8, RS = (TS * 5 + 3) / 4 * 4;
        d.Kp = Kp;
        std::vector<float> small((size_t)Kp * 20, 0.f), thp((size_t)Kp * 12, 0.f), BW((size_t)4 * Kp * 16, 1.f);
        std::vector<double> h0p((size_t)Kp * 2, 0.0);
        std::vector<float> dt((size_t)36 * TS * RS, 0.f);
        for (int k = 0; k < Kp; ++k) {
            float* sp = &small[(size_t)k * 20];
            if (k < K) {
                sp[0] = t.invW[k];
                sp[1] = t.sqrtW[k];
                for (int m = 0; m < 5; ++m) {
                    sp[2 + m] = t.visc[k * 5 + m];
                    sp[7 + m] = t.cond[k * 5 + m];
                    sp[12 + m] = t.ddiag[k * 5 + m];
                }
                for (int i = 0; i < 12; ++i) thp[(size_t)k * 12 + i] = t.th32[(size_t)k * 12 + i];
                h0p[k * 2] = t.th64[(size_t)(k * 2) * 6];
                h0p[k * 2 + 1] = t.th64[(size_t)(k * 2 + 1) * 6];
            } else {
                sp[2] = 1.f;   // g = 1
                sp[7] = 1.f;   // lambda_k = 1 (X_k = 0 anyway)
                sp[12] = 1.f;
            }
        }
        for (int w = 0; w < 4; ++w)
            for (int j = 0; j < K; ++j)
                for (int a = 0; a < KW; ++a) {
                    const int k = w * KW + a;
                    if (k < K) BW[((size_t)w * Kp + j) * 16 + a] = t.wilkeB[(size_t)k * K + j];
                }
        // Wilke's B factored (common.cuh): B = U diag(s) V^T from the fp64 weights, truncated after kWilkeRank terms, accepted
        // when every element of the truncated product is within 1e-6 of B (relative) and the factored form is cheaper
        std::vector<float> VW, UW;
        if (K > 28) {
            std::vector<double> A((size_t)K * K), Bd((size_t)K * K), V, sv;
            for (int k = 0; k < K; ++k)
                for (int j = 0; j < K; ++j) Bd[(size_t)k * K + j] = 1.0 / sqrt(8.0 * (1.0 + W[k] / W[j]));
            A = Bd;
            jacobi_svd(K, A, V, sv);   // A = U diag(s)
            int rank = 0;
            for (int r = 8; r <= kWilkeRank && !rank; r += 4) {   // the smallest of 8, 12 terms that reproduces every element to 1e-6
                double worst = 0.0;
                for (int k = 0; k < K; ++k)
                    for (int j = 0; j < K; ++j) {
                        double acc = 0.0;
                        for (int m = 0; m < r; ++m) acc += A[(size_t)k * K + m] * V[(size_t)j * K + m];
                        worst = fmax(worst, fabs(acc / Bd[(size_t)k * K + j] - 1.0));
                    }
                if (worst <= 1e-6) rank = r;
            }
            if (rank) {
                // the leading pair of singular vectors of a positive matrix has one sign: make it +, so that the m = 0 term
                // of a denominator is positive (the padding rows' denominators consist of it alone)
                double sg = 0.0;
                for (int j = 0; j < K; ++j) sg += V[(size_t)j * K];
                const double flip = sg < 0.0 ? -1.0 : 1.0;
                VW.assign((size_t)4 * Kp * 4, 0.f);
                UW.assign((size_t)4 * kWilkeRank * 16, 0.f);
                for (int w = 0; w < 4; ++w) {
                    for (int j = 0; j < K; ++j)
                        for (int c = 0; c < 3; ++c) {
                            const int m = w + 4 * c;
                            if (m < rank) VW[((size_t)w * Kp + j) * 4 + c] = (float)((m == 0 ? flip : 1.0) * V[(size_t)j * K + m]);
                        }
                    for (int m = 0; m < kWilkeRank; ++m)
                        for (int a = 0; a < KW; ++a) {
                            const int k = w * KW + a;
                            UW[((size_t)w * kWilkeRank + m) * 16 + a] =
                                k < K ? (float)((m == 0 ? flip : 1.0) * A[(size_t)k * K + m]) : (m == 0 ? 1.f : 0.f);
                        }
                }
                d.wilke_rank = rank;
            }
        }
        // eight species tiles of TS; tile pair (kt <= jt) number kt*8 - kt(kt-1)/2 + (jt - kt): [a][b][5], rows padded to RS
        size_t tix = 0;
        for (int kt = 0; kt < 8; ++kt)
            for (int jt = kt; jt < 8; ++jt, ++tix)
                for (int a = 0; a < TS; ++a)
                    for (int b = 0; b < TS; ++b) {
                        float* c = &dt[(tix * TS + a) * RS + (size_t)b * 5];
                        const int k = kt * TS + a, j = jt * TS + b;
                        if (k < K && j < K)
                            for (int m = 0; m < 5; ++m) c[m] = t.dfull[((size_t)k * K + j) * 5 + m];
                        else
                            c[0] = 1.f;
                    }
        if ((st = to_device(&d.small_p, small)) || (st = to_device(&d.thp, thp)) || (st = to_device(&d.h0p, h0p)) ||
            (st = to_device(&d.BW, BW)) || (st = to_device(&d.dtile, dt)) || (st = to_device(&d.VW, VW)) || (st = to_device(&d.UW, UW))) {
            df_mech_destroy(mech);
            return st;
        }
    }
    if (K == 9) mech->t9 = make_fixed<9>(t, W);
    if (K == 19) mech->t19 = make_fixed<19>(t, W);
    *out = mech;
    return DF_OK;
}

extern "C" df_status df_mech_destroy(df_mech* mech) {
    if (!mech) return DF_OK;
    MechDev& d = mech->dev;
    cudaFree(d.th32);
    cudaFree(d.sth32);
    cudaFree(d.th64);
    cudaFree(d.invW);
    cudaFree(d.sqrtW);
    cudaFree(d.visc);
    cudaFree(d.cond);
    cudaFree(d.ddiag);
    cudaFree(d.dfull);
    cudaFree(d.wilkeB);
    cudaFree(d.small_p);
    cudaFree(d.thp);
    cudaFree(d.h0p);
    cudaFree(d.BW);
    cudaFree(d.VW);
    cudaFree(d.UW);
    cudaFree(d.dtile);
    delete mech->t9;
    delete mech->t19;
    delete mech;
    return DF_OK;
}

extern "C" int df_mech_num_species(const df_mech* mech) { return mech ? mech->K : -1; }

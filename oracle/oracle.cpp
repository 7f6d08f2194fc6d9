// oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, fp64 CPU statement of what the hot path computes, written from the paper
// (/root/reference/PAPER.md, cited "P:line") and from the rule names BASELINE.json's
// north_star fixes where the paper is silent (readings A1..A20 in DESIGN.md / SURVEY.md 8(c)).
// It is the textbook loop nest: no mixture-polynomial collapse, no shifted variables, no
// rewritten Wilke sums, no blocking.  It shares no code, header, table or constant generator
// with paper_2312_05800_b200/csrc/ and neither includes the other.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load this library.  Parity pins: tests/test_oracle_*.py (every function below is
// pinned by a closed form, an invariant or brute force; nothing is "parity unpinned").
//
// The `#pragma omp parallel for` on the per-cell drivers is the only concession to speed:
// cells are independent ("computation of thermal and transport properties" is
// per cell; P:79 the ANN is applied per cell).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double R = 8314.46261815324;  // J/(kmol K)  (A1)

struct Mech {
    int K;
    std::vector<double> W, lo, hi, visc, cond, bdiff;
    double T_low, T_mid, T_high;
};

struct Ann {
    int n_layers;
    std::vector<int> dims;
    std::vector<std::vector<double>> W, b;
    std::vector<double> x_mean, x_std, u_mean, u_std;
    double lambda, dt;
};

// O1 -- NASA-7, two ranges, `hi` for T >= T_mid (A2), plain extrapolation outside (A3).
// cp_k/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
// h_k/(R T) = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T
// s_k/R = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7          (molar, J/kmol(/K))
void species_thermo(const Mech& m, int k, double T, double* cp, double* h, double* s) {
    const double* a = (T < m.T_mid ? m.lo.data() : m.hi.data()) + 7 * k;
    const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    if (cp) *cp = R * (a[0] + a[1] * T + a[2] * T2 + a[3] * T3 + a[4] * T4);
    if (h) *h = R * T * (a[0] + a[1] * T / 2.0 + a[2] * T2 / 3.0 + a[3] * T3 / 4.0 + a[4] * T4 / 5.0 + a[5] / T);
    if (s) *s = R * (a[0] * std::log(T) + a[1] * T + a[2] * T2 / 2.0 + a[3] * T3 / 3.0 + a[4] * T4 / 4.0 + a[6]);
}

// O2 -- mass-specific mixture cp = sum Y_k cp_k / W_k, h = sum Y_k h_k / W_k.
void mixture_cp_h(const Mech& m, double T, const double* Y, long long ld, double* cp, double* h) {
    double c = 0.0, e = 0.0;
    for (int k = 0; k < m.K; ++k) {
        double ck, hk;
        species_thermo(m, k, T, &ck, &hk, nullptr);
        c += Y[k * ld] * ck / m.W[k];
        e += Y[k * ld] * hk / m.W[k];
    }
    *cp = c;
    *h = e;
}

// O3 -- Newton on h(T, Y) = h_in:  T <- T - (h(T,Y) - h_in)/cp(T,Y)   (A4).
double newton_T(const Mech& m, double h_in, const double* Y, long long ld, double guess, int* iters) {
    double T = (std::isfinite(guess) && guess > 0.0) ? guess : m.T_mid;
    int it = 0;
    for (; it < 100; ++it) {
        double cp, h;
        mixture_cp_h(m, T, Y, ld, &cp, &h);
        const double delta = (h - h_in) / cp;
        T -= delta;
        if (T < 50.0) T = 50.0;
        if (T > 6000.0) T = 6000.0;
        if (std::fabs(delta) < 1e-9) { ++it; break; }
    }
    if (iters) *iters = it;
    return T;
}

double poly4(const double* c, double L) {
    return c[0] + c[1] * L + c[2] * L * L + c[3] * L * L * L + c[4] * L * L * L * L;
}

// O5 -- pure-species transport from the fits (A5), L = ln T:
// mu_k = sqrt(T) (sum b_m L^m)^2 ; lambda_k = sqrt(T) sum c_m L^m ; D_jk = T^{3/2} (sum d_m L^m) / p.
void species_transport(const Mech& m, double T, double p, double* mu, double* lam, double* D) {
    const int K = m.K;
    const double L = std::log(T);
    for (int k = 0; k < K; ++k) {
        const double q = poly4(&m.visc[5 * k], L);
        if (mu) mu[k] = std::sqrt(T) * q * q;
        if (lam) lam[k] = std::sqrt(T) * poly4(&m.cond[5 * k], L);
    }
    if (D)
        for (int j = 0; j < K; ++j)
            for (int k = 0; k < K; ++k)
                D[j * K + k] = std::pow(T, 1.5) * poly4(&m.bdiff[5 * (j * K + k)], L) / p;
}

// O4, O6, O7, O8 for one cell.
void cell_properties(const Mech& m, double T, double p, const double* Y, long long ld,
                     double* cp, double* h, double* mu_out, double* lam_out, double* D_out, long long ldD) {
    const int K = m.K;
    std::vector<double> X(K), mu(K), lam(K), D(K * K);
    // O4: X_k = (Y_k/W_k) / sum_j (Y_j/W_j); Y used as given.
    double inv_Wbar = 0.0;
    for (int k = 0; k < K; ++k) inv_Wbar += Y[k * ld] / m.W[k];
    for (int k = 0; k < K; ++k) X[k] = (Y[k * ld] / m.W[k]) / inv_Wbar;
    if (cp || h) {
        double c, e;
        mixture_cp_h(m, T, Y, ld, &c, &e);
        if (cp) *cp = c;
        if (h) *h = e;
    }
    species_transport(m, T, p, mu.data(), lam.data(), D.data());
    // O6: Wilke.  mu = sum_k X_k mu_k / sum_j X_j Phi_kj,
    // Phi_kj = [1 + (mu_k/mu_j)^{1/2} (W_j/W_k)^{1/4}]^2 / [8 (1 + W_k/W_j)]^{1/2}.
    if (mu_out) {
        double s = 0.0;
        for (int k = 0; k < K; ++k) {
            double den = 0.0;
            for (int j = 0; j < K; ++j) {
                const double a = 1.0 + std::sqrt(mu[k] / mu[j]) * std::pow(m.W[j] / m.W[k], 0.25);
                const double phi = a * a / std::sqrt(8.0 * (1.0 + m.W[k] / m.W[j]));
                den += X[j] * phi;
            }
            s += X[k] * mu[k] / den;
        }
        *mu_out = s;
    }
    // O7: combination rule lambda = 1/2 [ sum X_k lambda_k + 1 / sum (X_k / lambda_k) ]   (A6).
    if (lam_out) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < K; ++k) {
            a += X[k] * lam[k];
            b += X[k] / lam[k];
        }
        *lam_out = 0.5 * (a + 1.0 / b);
    }
    // O8: D_km = sum_{j != k} Y_j / sum_{j != k} X_j / D_jk, self-diffusion if the mixture is pure k (A7).
    if (D_out)
        for (int k = 0; k < K; ++k) {
            double num = 0.0, den = 0.0;
            for (int j = 0; j < K; ++j) {
                if (j == k) continue;
                num += Y[j * ld];
                den += X[j] / D[j * K + k];
            }
            D_out[k * ldD] = den > 0.0 ? num / den : D[k * K + k];
        }
}

// P:79 "The Box-Cox transformation F(x) [25]"; formula from Box & Cox, lambda from the config (A10).
double boxcox(double y, double lambda) { return (std::pow(y, lambda) - 1.0) / lambda; }
double boxcox_inv(double f, double lambda) { return std::pow(lambda * f + 1.0, 1.0 / lambda); }

// P:79 "The Gaussian Error Linear Unit (GELU)": exact form x Phi(x) (A13), with the normal CDF written
// Phi(x) = erfc(-x/sqrt 2)/2, which is 1/2 (1 + erf(x/sqrt 2)) without the cancellation at x << 0.
double gelu(double x) { return x * 0.5 * std::erfc(-x / std::sqrt(2.0)); }

// O9 -- P:79 "x(t) {T(t), p(t), F(Y(t))}" then "Z-score normalization" (A8).
void cell_features(const Ann& a, double T, double p, const double* Y, long long ld, double* f) {
    const int K = a.dims.back();
    f[0] = (T - a.x_mean[0]) / a.x_std[0];
    f[1] = (p - a.x_mean[1]) / a.x_std[1];
    for (int k = 0; k < K; ++k) f[2 + k] = (boxcox(Y[k * ld], a.lambda) - a.x_mean[2 + k]) / a.x_std[2 + k];
}

// O10 -- P:79 "hidden layers with 1600, 800, and 400 perceptrons ... GELU": naive loops,
// a_{l+1} = GELU(a_l W_l^T + b_l) on hidden layers, linear last layer; activations never rounded.
void mlp_forward(const Ann& a, const double* x, double* out) {
    std::vector<double> cur(x, x + a.dims[0]), nxt;
    for (int l = 0; l < a.n_layers; ++l) {
        const int din = a.dims[l], dout = a.dims[l + 1];
        nxt.assign(dout, 0.0);
        for (int o = 0; o < dout; ++o) {
            double acc = 0.0;
            for (int i = 0; i < din; ++i) acc += cur[i] * a.W[l][(size_t)o * din + i];
            acc += a.b[l][o];
            nxt[o] = (l + 1 < a.n_layers) ? gelu(acc) : acc;
        }
        cur.swap(nxt);
    }
    std::memcpy(out, cur.data(), sizeof(double) * a.dims.back());
}

// O11/O12 -- output is the z-scored change in Box-Cox space (A9): Delta_k = s^u_k o_k + m^u_k,
// Y*_k = max(Y_k^lambda + lambda Delta_k, 0)^{1/lambda} (A10), Y' = Y*/sum Y* (A11, "mass
// fractions ... must sum to unity"), dY = Y' - Y over dt ("time step of 1 us"),
// rho = p Wbar/(R T) (A17), omega_k = rho dY_k / dt.
void cell_source(const Ann& a, const Mech& m, double T, double p, const double* Y, long long ld,
                 double* omega, double* dY, long long ldo) {
    const int K = m.K;
    std::vector<double> f(K + 2), o(K), Ys(K);
    cell_features(a, T, p, Y, ld, f.data());
    mlp_forward(a, f.data(), o.data());
    double S = 0.0;
    for (int k = 0; k < K; ++k) {
        const double delta = a.u_std[k] * o[k] + a.u_mean[k];
        double base = std::pow(Y[k * ld], a.lambda) + a.lambda * delta;
        if (base < 0.0) base = 0.0;
        Ys[k] = std::pow(base, 1.0 / a.lambda);
        S += Ys[k];
    }
    double inv_Wbar = 0.0;
    for (int k = 0; k < K; ++k) inv_Wbar += Y[k * ld] / m.W[k];
    const double rho = p / (inv_Wbar * R * T);
    for (int k = 0; k < K; ++k) {
        const double d = Ys[k] / S - Y[k * ld];
        if (dY) dY[k * ldo] = d;
        if (omega) omega[k * ldo] = rho * d / a.dt;
    }
}

// ---- NEXT-1: one MLP per species --------------------------------------------------------------------
// P:79 "individual training and prediction are carried out for each species mass fraction" ("multiple multilayer
// perceptrons"): K independent networks (K+2) -> ... -> 1 share the input vector x = {T, p, F(Y)} (O9) and each
// predicts the z-scored Box-Cox-space change of ITS species: Delta_k = s^u_k o^(k) + m^u_k (A9).  Everything after the
// networks is O11/O12 exactly as in cell_source (inverse Box-Cox with base clamp A10, Y' = Y*/sum Y* A11, ideal-gas
// rho A17).  nets[k] is an Ann with dims[0] = K + 2 and one output; its x_mean/x_std are the shared input statistics
// (taken from nets[0]), its u_mean[0]/u_std[0] are species k's.
void cell_source_mmlp(const Ann* const* nets, const Mech& m, double T, double p, const double* Y, long long ld,
                      double* omega, double* dY, long long ldo) {
    const int K = m.K;
    const Ann& a0 = *nets[0];
    std::vector<double> f(K + 2), Ys(K);
    f[0] = (T - a0.x_mean[0]) / a0.x_std[0];
    f[1] = (p - a0.x_mean[1]) / a0.x_std[1];
    for (int k = 0; k < K; ++k) f[2 + k] = (boxcox(Y[k * ld], a0.lambda) - a0.x_mean[2 + k]) / a0.x_std[2 + k];
    double S = 0.0;
    for (int k = 0; k < K; ++k) {
        double o;
        mlp_forward(*nets[k], f.data(), &o);
        const double delta = nets[k]->u_std[0] * o + nets[k]->u_mean[0];
        double base = std::pow(Y[k * ld], a0.lambda) + a0.lambda * delta;
        if (base < 0.0) base = 0.0;
        Ys[k] = std::pow(base, 1.0 / a0.lambda);
        S += Ys[k];
    }
    double inv_Wbar = 0.0;
    for (int k = 0; k < K; ++k) inv_Wbar += Y[k * ld] / m.W[k];
    const double rho = p / (inv_Wbar * R * T);
    for (int k = 0; k < K; ++k) {
        const double d = Ys[k] / S - Y[k * ld];
        if (dY) dY[k * ldo] = d;
        if (omega) omega[k * ldo] = rho * d / a0.dt;
    }
}

// ---- NEXT-4: solver-facing extras of the property pass -------------------------------------------
// P:34-36 "computation of thermal and transport properties" for a compressible solver with non-unity Lewis numbers
// ("Hirschfelder and Curtiss mixture-averaged transport"): besides cp, h, mu, lambda, D_k the transport
// equations need rho, psi = d rho / d p at constant T, alpha = lambda / cp, rho D_k, the species enthalpies h_k(T)
// of the diffusive enthalpy flux sum_k h_k J_k, and (for diagnostics) the mixture entropy.  Reading A22:
//   rho = p Wbar / (R T)   psi = Wbar / (R T)   alpha = lambda / cp   (rho D)_k = rho D_k   h_k = h_k(T) / W_k  [J/kg]
//   s = sum_k (Y_k / W_k) [ s_k(T) - R ln X_k ] - (R / Wbar) ln(p / p0),  p0 = 101325 Pa, terms with X_k = 0 drop out
// (ideal-gas mixture: standard-state species entropies O1, entropy of mixing, pressure correction).
constexpr double P0 = 101325.0;
void cell_extras(const Mech& m, double T, double p, const double* Y, long long ld, double cp, double lam, const double* D,
                 long long ldD, double* rho_o, double* psi_o, double* alpha_o, double* rhoD, double* hk, long long ldo,
                 double* s_o) {
    const int K = m.K;
    double inv_Wbar = 0.0;
    for (int k = 0; k < K; ++k) inv_Wbar += Y[k * ld] / m.W[k];
    const double Wbar = 1.0 / inv_Wbar;
    const double rho = p * Wbar / (R * T);
    if (rho_o) *rho_o = rho;
    if (psi_o) *psi_o = Wbar / (R * T);
    if (alpha_o) *alpha_o = lam / cp;
    double s = 0.0;
    for (int k = 0; k < K; ++k) {
        double hkm, sk;
        species_thermo(m, k, T, nullptr, &hkm, &sk);
        if (hk) hk[k * ldo] = hkm / m.W[k];
        if (rhoD) rhoD[k * ldo] = rho * D[k * ldD];
        const double X = (Y[k * ld] / m.W[k]) * Wbar;
        if (X > 0.0) s += (Y[k * ld] / m.W[k]) * (sk - R * std::log(X));
    }
    s -= (R / Wbar) * std::log(p / P0);
    if (s_o) *s_o = s;
}

// ---- NEXT-3: PaSR scaling of the ANN source and the temperature gate ------------------------------
// P:113 "the PaSR combustion model wherein the characteristic chemical time is calculated as the slowest formation
// rate of species and the mixing time scale is calculated as the geometric mean of the Taylor scale and the
// Kolmogorov scale"; "a minimum temperature threshold of 500 K" (the ANN was never shown colder states).
// The paper prints no formula.  Reading A23:
//   tau_c   = max over species with |omega_k| > 0 of rho Y_k / |omega_k|      (slowest species time scale; 0 if none)
//   tau_mix = sqrt( (k_sgs / eps) * sqrt(nu / eps) ),  nu = mu / rho           (Taylor x Kolmogorov time scales)
//   kappa   = tau_c / (tau_c + tau_mix)   (0 when tau_c = 0);   omega_k <- kappa omega_k;   T < T_gate => omega_k <- 0
void cell_pasr(const Mech& m, double T, double p, const double* Y, long long ld, double mu, double ksgs, double eps,
               double T_gate, const double* om_in, double* om_out, long long ldo, double* kappa_o) {
    const int K = m.K;
    double inv_Wbar = 0.0;
    for (int k = 0; k < K; ++k) inv_Wbar += Y[k * ld] / m.W[k];
    const double rho = p / (inv_Wbar * R * T);
    double tau_c = 0.0;
    for (int k = 0; k < K; ++k) {
        const double w = std::fabs(om_in[k * ldo]);
        if (w > 0.0) tau_c = std::max(tau_c, rho * Y[k * ld] / w);
    }
    const double tau_mix = std::sqrt((ksgs / eps) * std::sqrt((mu / rho) / eps));
    double kappa = tau_c > 0.0 ? tau_c / (tau_c + tau_mix) : 0.0;
    if (T < T_gate) kappa = 0.0;
    for (int k = 0; k < K; ++k) om_out[k * ldo] = kappa * om_in[k * ldo];
    if (kappa_o) *kappa_o = kappa;
}

}  // namespace

extern "C" {

void* oracle_mech_create(int K, const double* W, const double* nasa_lo, const double* nasa_hi,
                         double T_low, double T_mid, double T_high,
                         const double* visc_fit, const double* cond_fit, const double* bdiff_fit) {
    Mech* m = new Mech;
    m->K = K;
    m->W.assign(W, W + K);
    m->lo.assign(nasa_lo, nasa_lo + 7 * K);
    m->hi.assign(nasa_hi, nasa_hi + 7 * K);
    m->visc.assign(visc_fit, visc_fit + 5 * K);
    m->cond.assign(cond_fit, cond_fit + 5 * K);
    m->bdiff.assign(bdiff_fit, bdiff_fit + 5 * (size_t)K * K);
    m->T_low = T_low;
    m->T_mid = T_mid;
    m->T_high = T_high;
    return m;
}
void oracle_mech_destroy(void* m) { delete static_cast<Mech*>(m); }

void* oracle_ann_create(int n_layers, const int* dims, const double* W_flat, const double* b_flat,
                        const double* x_mean, const double* x_std, const double* u_mean, const double* u_std,
                        double lambda, double dt) {
    Ann* a = new Ann;
    a->n_layers = n_layers;
    a->dims.assign(dims, dims + n_layers + 1);
    size_t wo = 0, bo = 0;
    for (int l = 0; l < n_layers; ++l) {
        const size_t nw = (size_t)dims[l] * dims[l + 1];
        a->W.emplace_back(W_flat + wo, W_flat + wo + nw);
        a->b.emplace_back(b_flat + bo, b_flat + bo + dims[l + 1]);
        wo += nw;
        bo += dims[l + 1];
    }
    const int K = dims[n_layers];
    a->x_mean.assign(x_mean, x_mean + dims[0]);
    a->x_std.assign(x_std, x_std + dims[0]);
    a->u_mean.assign(u_mean, u_mean + K);
    a->u_std.assign(u_std, u_std + K);
    a->lambda = lambda;
    a->dt = dt;
    return a;
}
void oracle_ann_destroy(void* a) { delete static_cast<Ann*>(a); }

void oracle_set_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n > 0 ? n : 1);
#else
    (void)n;
#endif
}
int oracle_get_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_species_thermo(const void* m, int k, double T, double* cp, double* h, double* s) {
    species_thermo(*static_cast<const Mech*>(m), k, T, cp, h, s);
}

void oracle_species_transport(const void* m, double T, double p, double* mu_k, double* lambda_k, double* D_jk) {
    species_transport(*static_cast<const Mech*>(m), T, p, mu_k, lambda_k, D_jk);
}

void oracle_mixture_cp_h(const void* mv, long long n, long long ld, const double* T, const double* Y,
                         double* cp, double* h) {
    const Mech& m = *static_cast<const Mech*>(mv);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i) mixture_cp_h(m, T[i], Y + i, ld, &cp[i], &h[i]);
}

void oracle_T_from_h(const void* mv, long long n, long long ld, const double* h, const double* Y,
                     const double* T_guess, double* T_out, int* iters) {
    const Mech& m = *static_cast<const Mech*>(mv);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i) T_out[i] = newton_T(m, h[i], Y + i, ld, T_guess[i], iters ? &iters[i] : nullptr);
}

void oracle_properties(const void* mv, long long n, long long ld, const double* T, const double* p, const double* Y,
                       double* cp, double* h, double* mu, double* lambda, double* D) {
    const Mech& m = *static_cast<const Mech*>(mv);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i)
        cell_properties(m, T[i], p[i], Y + i, ld, cp ? &cp[i] : nullptr, h ? &h[i] : nullptr,
                        mu ? &mu[i] : nullptr, lambda ? &lambda[i] : nullptr, D ? D + i : nullptr, ld);
}

double oracle_boxcox(double y, double lambda) { return boxcox(y, lambda); }
double oracle_boxcox_inv(double f, double lambda) { return boxcox_inv(f, lambda); }
double oracle_gelu(double x) { return gelu(x); }

void oracle_ann_features(const void* av, long long n, long long ld, const double* T, const double* p, const double* Y,
                         double* f) {
    const Ann& a = *static_cast<const Ann*>(av);
    const int d0 = a.dims[0];
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i) cell_features(a, T[i], p[i], Y + i, ld, f + i * d0);
}

void oracle_mlp_forward(const void* av, long long n, const double* x, double* out) {
    const Ann& a = *static_cast<const Ann*>(av);
    const int d0 = a.dims[0], dL = a.dims.back();
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i) mlp_forward(a, x + i * d0, out + i * dL);
}

void oracle_ann_source(const void* av, const void* mv, long long n, long long ld, const double* T, const double* p,
                       const double* Y, double* omega, double* dY) {
    const Ann& a = *static_cast<const Ann*>(av);
    const Mech& m = *static_cast<const Mech*>(mv);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i)
        cell_source(a, m, T[i], p[i], Y + i, ld, omega ? omega + i : nullptr, dY ? dY + i : nullptr, ld);
}

void oracle_extras(const void* mv, long long n, long long ld, const double* T, const double* p, const double* Y,
                   const double* cp, const double* lam, const double* D, double* rho, double* psi, double* alpha,
                   double* rhoD, double* hk, double* s) {
    const Mech& m = *static_cast<const Mech*>(mv);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i)
        cell_extras(m, T[i], p[i], Y + i, ld, cp ? cp[i] : 1.0, lam ? lam[i] : 0.0, D ? D + i : nullptr, ld,
                    rho ? &rho[i] : nullptr, psi ? &psi[i] : nullptr, (alpha && cp && lam) ? &alpha[i] : nullptr,
                    (rhoD && D) ? rhoD + i : nullptr, hk ? hk + i : nullptr, ld, s ? &s[i] : nullptr);
}

void oracle_pasr(const void* mv, long long n, long long ld, const double* T, const double* p, const double* Y,
                 const double* mu, const double* ksgs, const double* eps, double T_gate, const double* om_in,
                 double* om_out, double* kappa) {
    const Mech& m = *static_cast<const Mech*>(mv);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i)
        cell_pasr(m, T[i], p[i], Y + i, ld, mu[i], ksgs[i], eps[i], T_gate, om_in + i, om_out + i, ld,
                  kappa ? &kappa[i] : nullptr);
}

void oracle_ann_source_mmlp(const void* const* nets, const void* mv, long long n, long long ld, const double* T,
                            const double* p, const double* Y, double* omega, double* dY) {
    const Mech& m = *static_cast<const Mech*>(mv);
    const Ann* const* a = reinterpret_cast<const Ann* const*>(nets);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < n; ++i)
        cell_source_mmlp(a, m, T[i], p[i], Y + i, ld, omega ? omega + i : nullptr, dY ? dY + i : nullptr, ld);
}

}  // extern "C"

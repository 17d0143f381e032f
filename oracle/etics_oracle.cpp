// etics_oracle.cpp — CPU ORACLE for the ETICS expansion force calculation.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
// header, table or constant generator with the CUDA path under paper_1406_4254_b200/csrc/.
//
// What it is: a plain, slow, one-particle-at-a-time fp64 restatement of the two truncated series the
// paper evaluates (both are truncated expansions, not accelerations of an exact result, so the oracle
// is the algorithm itself, written in the paper's order and notation):
//   * SCF  — eq. (18) PAPER.md:161 (§2.4), with the Hernquist–Ostriker (HO92) radial basis the paper
//            adopts (§2.5, §5.1); two parts as in PAPER.md:217-219 (§3.3):
//            (1) all A_nlm from the particles, (2) force/potential of every particle from the A_nlm.
//   * MEX  — eqs. (15)–(17) PAPER.md:146-155 (§2.4) with the discrete *exclusive* cumulative sums of
//            eqs. (11)–(12) PAPER.md:120-123 and the radial sort of PAPER.md:157, 207.
// Real form throughout: A_nlm (cos m phi) and B_nlm (sin m phi), m >= 0 (the paper's complex
// coefficients for -m are complex conjugates).  G = 1, a = 1, centre = origin.
//
// The HO92 formulas themselves are NOT printed in PAPER.md (it cites HO92); the forms used here are
// listed in DESIGN.md "Readings" (G1) and are pinned — independently of this file — by
// tests/test_oracle_pins_*.py (Poisson identity, biorthogonality by exact quadrature, analytic
// Hernquist potential, pairwise addition-theorem identities, brute-force Newtonian sums).
// Parity status: every exported function below has at least one such pin; none is "parity unpinned".
//
// Every sum over particles uses Neumaier compensated summation so that the oracle's own rounding is
// far below the 1e-10 parity tolerance.  Compile with -O2 -ffp-contract=off (oracle/build.py) so that
// no FMA contraction happens except where std::fma is written out (the sort key, reading G7).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double PI = 3.14159265358979323846264338327950288;

struct Neumaier {
    double s = 0.0, c = 0.0;
    inline void add(double x) {
        double t = s + x;
        if (std::fabs(s) >= std::fabs(x)) c += (s - t) + x; else c += (x - t) + s;
        s = t;
    }
    inline double value() const { return s + c; }
};

inline int lm_index(int l, int m) { return l * (l + 1) / 2 + m; }
inline int num_lm(int lmax) { return (lmax + 1) * (lmax + 2) / 2; }

// ---------------------------------------------------------------------------------------------
// Per-particle geometry (SURVEY.md §8(c) "Common per-particle functions").
// On-axis particles (x = y = 0) are legal: phi := 0 (reading G10).
// ---------------------------------------------------------------------------------------------
struct Geom { double r, ct, st, cp, sp; };

inline Geom geometry(double x, double y, double z) {
    Geom g;
    double rho2 = x * x + y * y;
    double rho = std::sqrt(rho2);
    g.r = std::sqrt(rho2 + z * z);
    g.ct = z / g.r;
    g.st = rho / g.r;
    if (rho > 0.0) { g.cp = x / rho; g.sp = y / rho; } else { g.cp = 1.0; g.sp = 0.0; }
    return g;
}

// cos(m phi), sin(m phi), m = 0..lmax, by angle addition.
inline void trig_table(int lmax, double cp, double sp, double* cm, double* sm) {
    cm[0] = 1.0; sm[0] = 0.0;
    for (int m = 1; m <= lmax; ++m) {
        cm[m] = cm[m - 1] * cp - sm[m - 1] * sp;
        sm[m] = sm[m - 1] * cp + cm[m - 1] * sp;
    }
}

// ---------------------------------------------------------------------------------------------
// Associated Legendre functions P_l^m(cos theta) WITHOUT the Condon–Shortley phase (P_11 = +sin),
// by the l-recurrence that is stable near the poles; the paper's own m-recurrence, eq. (24)
// PAPER.md:346-350, is what the paper itself blames for its single-precision errors and is not used.
//   P_mm = (2m-1)!! sin^m;  P_{m+1,m} = (2m+1) cos P_mm;
//   (l-m) P_lm = (2l-1) cos P_{l-1,m} - (l+m-1) P_{l-2,m}.
// U_lm = P_lm / sin(theta) for m >= 1 comes from the SAME recurrence seeded with
// U_mm = (2m-1)!! sin^(m-1) (a polynomial: nothing is ever divided by sin theta).  U_l0 := 0 (unused).
// dP_lm/dtheta = 1/2 [ (l+m)(l-m+1) P_{l,m-1} - P_{l,m+1} ],  P_{l,-1} = -P_{l,1}/(l(l+1)), P_{l,l+1} = 0.
// Packed index lm_index(l,m), 0 <= m <= l <= lmax.
// ---------------------------------------------------------------------------------------------
void legendre_table(int lmax, double ct, double st, double* P, double* dP, double* U) {
    double dfact = 1.0;      // (2m-1)!!
    double spow = 1.0;       // sin^m
    double spow1 = 0.0;      // sin^(m-1) (m >= 1)
    for (int m = 0; m <= lmax; ++m) {
        if (m > 0) {
            dfact *= (2 * m - 1);
            spow1 = spow;
            spow *= st;
        }
        double pmm = dfact * spow;
        double umm = (m > 0) ? dfact * spow1 : 0.0;
        P[lm_index(m, m)] = pmm;
        U[lm_index(m, m)] = umm;
        if (m + 1 <= lmax) {
            P[lm_index(m + 1, m)] = (2 * m + 1) * ct * pmm;
            U[lm_index(m + 1, m)] = (2 * m + 1) * ct * umm;
        }
        for (int l = m + 2; l <= lmax; ++l) {
            P[lm_index(l, m)] = ((2 * l - 1) * ct * P[lm_index(l - 1, m)] - (l + m - 1) * P[lm_index(l - 2, m)]) / (l - m);
            U[lm_index(l, m)] = ((2 * l - 1) * ct * U[lm_index(l - 1, m)] - (l + m - 1) * U[lm_index(l - 2, m)]) / (l - m);
        }
    }
    for (int l = 0; l <= lmax; ++l) {
        for (int m = 0; m <= l; ++m) {
            double below, above;
            if (m == 0) below = (l > 0) ? -P[lm_index(l, 1)] / (double(l) * (l + 1)) : 0.0;
            else below = P[lm_index(l, m - 1)];
            above = (m + 1 <= l) ? P[lm_index(l, m + 1)] : 0.0;
            dP[lm_index(l, m)] = 0.5 * (double(l + m) * (l - m + 1) * below - above);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Gegenbauer (ultraspherical) polynomials C_n^(alpha)(xi), n = 0..nmax, and d/dxi by
// differentiating the three-term recurrence (the paper's "W_nl", reading G6):
//   C_0 = 1, C_1 = 2 alpha xi,  n C_n = 2(n+alpha-1) xi C_{n-1} - (n+2alpha-2) C_{n-2}.
// ---------------------------------------------------------------------------------------------
void gegenbauer_table(int nmax, double alpha, double xi, double* C, double* dC) {
    C[0] = 1.0; dC[0] = 0.0;
    if (nmax >= 1) { C[1] = 2.0 * alpha * xi; dC[1] = 2.0 * alpha; }
    for (int n = 2; n <= nmax; ++n) {
        double a = 2.0 * (n + alpha - 1.0), b = n + 2.0 * alpha - 2.0;
        C[n] = (a * xi * C[n - 1] - b * C[n - 2]) / n;
        dC[n] = (a * (C[n - 1] + xi * dC[n - 1]) - b * dC[n - 2]) / n;
    }
}

// ---------------------------------------------------------------------------------------------
// HO92 basis constants (reading G1).
//   K_nl = n(n+4l+3)/2 + (l+1)(2l+1)
//   I_nl = int_0^inf 4 pi rho~_nl Phi~_nl r^2 dr
//        = -K_nl * 4 pi / 2^(8l+6) * Gamma(n+4l+3) / ( n! (n+2l+3/2) Gamma(2l+3/2)^2 )
//   A~_nl = 4 pi / I_nl          (A~_00 = -12 pi, I_00 = -1/3)
//   N_lm = (2 - delta_m0) (2l+1)/(4 pi) (l-m)!/(l+m)!      (+-m folded into m >= 0)
//   w_lm = (2 - delta_m0) (l-m)!/(l+m)!                    (= N_lm 4 pi/(2l+1); MEX weight)
// ---------------------------------------------------------------------------------------------
double K_nl(int n, int l) { return 0.5 * n * (n + 4.0 * l + 3.0) + (l + 1.0) * (2.0 * l + 1.0); }

double I_nl(int n, int l) {
    long double lg = lgammal((long double)(n + 4 * l + 3)) - lgammal((long double)(n + 1))
                   - 2.0L * lgammal(2.0L * l + 1.5L) - (8.0L * l + 6.0L) * logl(2.0L);
    long double v = -(long double)K_nl(n, l) * 4.0L * (long double)PI * expl(lg) / ((long double)n + 2.0L * l + 1.5L);
    return (double)v;
}
double Atilde_nl(int n, int l) { return 4.0 * PI / I_nl(n, l); }

double fact_ratio(int l, int m) {   // (l-m)!/(l+m)!
    double v = 1.0;
    for (int k = l - m + 1; k <= l + m; ++k) v /= k;
    return v;
}
double w_lm(int l, int m) { return (m == 0 ? 1.0 : 2.0) * fact_ratio(l, m); }
double N_lm(int l, int m) { return w_lm(l, m) * (2 * l + 1) / (4.0 * PI); }

// ---------------------------------------------------------------------------------------------
// Radial basis: Phi~_nl(r) = -r^l/(1+r)^(2l+1) C_n^(2l+3/2)(xi),  xi = (r-1)/(r+1),
// and dPhi~_nl/dr.  Output index l*(nmax+1)+n.
//   f_l(r) = -r^l (1+r)^-(2l+1);  f_l'(r) = -( l r^(l-1) (1+r) - (2l+1) r^l ) (1+r)^-(2l+2);  dxi/dr = 2/(1+r)^2
// ---------------------------------------------------------------------------------------------
void radial_table(int nmax, int lmax, double r, double* Phi, double* dPhi) {
    std::vector<double> C(nmax + 1), dC(nmax + 1);
    double xi = (r - 1.0) / (r + 1.0);
    double dxi = 2.0 / ((1.0 + r) * (1.0 + r));
    for (int l = 0; l <= lmax; ++l) {
        double f = -std::pow(r, l) / std::pow(1.0 + r, 2 * l + 1);
        double lead = (l == 0) ? 0.0 : l * std::pow(r, l - 1) * (1.0 + r);
        double fp = -(lead - (2 * l + 1) * std::pow(r, l)) / std::pow(1.0 + r, 2 * l + 2);
        gegenbauer_table(nmax, 2.0 * l + 1.5, xi, C.data(), dC.data());
        for (int n = 0; n <= nmax; ++n) {
            Phi[l * (nmax + 1) + n] = f * C[n];
            dPhi[l * (nmax + 1) + n] = fp * C[n] + f * dC[n] * dxi;
        }
    }
}

// rho~_nl(r) = K_nl/(2 pi) r^l / ( r (1+r)^(2l+3) ) C_n^(2l+3/2)(xi)   (used only by the pins)
void density_table(int nmax, int lmax, double r, double* Rho) {
    std::vector<double> C(nmax + 1), dC(nmax + 1);
    double xi = (r - 1.0) / (r + 1.0);
    for (int l = 0; l <= lmax; ++l) {
        gegenbauer_table(nmax, 2.0 * l + 1.5, xi, C.data(), dC.data());
        double g = std::pow(r, l) / (r * std::pow(1.0 + r, 2 * l + 3)) / (2.0 * PI);
        for (int n = 0; n <= nmax; ++n) Rho[l * (nmax + 1) + n] = K_nl(n, l) * g * C[n];
    }
}

int resolve_threads(int threads) {
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
    return threads;
#else
    (void)threads;
    return 1;
#endif
}

// Spherical -> Cartesian ("transforms it to Cartesian coordinates").
inline void to_cartesian(const Geom& g, double ar, double at, double ap, double* ax, double* ay, double* az) {
    *ax = ar * g.st * g.cp + at * g.ct * g.cp - ap * g.sp;
    *ay = ar * g.st * g.sp + at * g.ct * g.sp + ap * g.cp;
    *az = ar * g.ct - at * g.st;
}

}  // namespace

extern "C" {

int oracle_num_threads(int threads) { return resolve_threads(threads); }

// ---- engines, exported so that the pins can test each one on its own ---------------------------
void oracle_gegenbauer(int nmax, double alpha, double xi, double* C, double* dC) { gegenbauer_table(nmax, alpha, xi, C, dC); }
void oracle_legendre(int lmax, double ct, double st, double* P, double* dP, double* U) { legendre_table(lmax, ct, st, P, dP, U); }
void oracle_radial(int nmax, int lmax, double r, double* Phi, double* dPhi) { radial_table(nmax, lmax, r, Phi, dPhi); }
void oracle_density(int nmax, int lmax, double r, double* Rho) { density_table(nmax, lmax, r, Rho); }
double oracle_K_nl(int n, int l) { return K_nl(n, l); }
double oracle_I_nl(int n, int l) { return I_nl(n, l); }
double oracle_Atilde_nl(int n, int l) { return Atilde_nl(n, l); }
double oracle_N_lm(int l, int m) { return N_lm(l, m); }
double oracle_w_lm(int l, int m) { return w_lm(l, m); }

// ---------------------------------------------------------------------------------------------
// SCF part (1): all coefficients (PAPER.md:217-219 step 1a/1b; eq. 18).
//   S^c_nlm = sum_k m_k Phi~_nl(r_k) P_lm(k) cos(m phi_k);  S^s_nlm with sin;
//   A_nlm = A~_nl N_lm S^c_nlm,  B_nlm = A~_nl N_lm S^s_nlm  (B_nl0 = +0).
// The particle's own contribution is included (a field method cannot exclude it; reading G9).
// pos = x[0..N) | y | z ; A, B have T = (nmax+1) L entries, index n*L + l(l+1)/2 + m.
// threads: OpenMP threads (<=0: all); thread-private tables are combined in thread order.
// ---------------------------------------------------------------------------------------------
int oracle_scf_coeffs(const double* pos, const double* mass, long long N, int nmax, int lmax,
                      double* A, double* B, int threads) {
    if (N < 1 || nmax < 0 || lmax < 0) return -1;
    const int L = num_lm(lmax), T = (nmax + 1) * L;
    threads = resolve_threads(threads);
    std::vector<std::vector<Neumaier>> Sc(threads, std::vector<Neumaier>(T)), Ss(threads, std::vector<Neumaier>(T));
    const double *X = pos, *Y = pos + N, *Z = pos + 2 * N;
#pragma omp parallel num_threads(threads)
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num();
#else
        const int tid = 0;
#endif
        std::vector<double> P(L), dP(L), U(L), cm(lmax + 1), sm(lmax + 1);
        std::vector<double> Phi((nmax + 1) * (lmax + 1)), dPhi((nmax + 1) * (lmax + 1));
        const long long k0 = N * tid / threads, k1 = N * (tid + 1) / threads;
        for (long long k = k0; k < k1; ++k) {
            Geom g = geometry(X[k], Y[k], Z[k]);
            legendre_table(lmax, g.ct, g.st, P.data(), dP.data(), U.data());
            trig_table(lmax, g.cp, g.sp, cm.data(), sm.data());
            radial_table(nmax, lmax, g.r, Phi.data(), dPhi.data());
            for (int n = 0; n <= nmax; ++n)
                for (int l = 0; l <= lmax; ++l)
                    for (int m = 0; m <= l; ++m) {
                        double t = mass[k] * Phi[l * (nmax + 1) + n] * P[lm_index(l, m)];
                        Sc[tid][n * L + lm_index(l, m)].add(t * cm[m]);
                        Ss[tid][n * L + lm_index(l, m)].add(t * sm[m]);
                    }
        }
    }
    for (int n = 0; n <= nmax; ++n)
        for (int l = 0; l <= lmax; ++l)
            for (int m = 0; m <= l; ++m) {
                Neumaier c, s;
                for (int t = 0; t < threads; ++t) {
                    c.add(Sc[t][n * L + lm_index(l, m)].s); c.add(Sc[t][n * L + lm_index(l, m)].c);
                    s.add(Ss[t][n * L + lm_index(l, m)].s); s.add(Ss[t][n * L + lm_index(l, m)].c);
                }
                double norm = Atilde_nl(n, l) * N_lm(l, m);
                A[n * L + lm_index(l, m)] = norm * c.value();
                B[n * L + lm_index(l, m)] = (m == 0) ? 0.0 : norm * s.value();
            }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// SCF part (2): potential and acceleration of every point from the coefficients
// (PAPER.md:219 step 2a/2b).  With E = A cos(m phi) + B sin(m phi),
// F = m(-A sin(m phi) + B cos(m phi)):
//   Phi   =       sum Phi~_nl        P_lm       E
//   a_r   = -     sum dPhi~_nl/dr    P_lm       E
//   a_th  = -1/r  sum Phi~_nl        dP_lm/dth  E
//   a_phi = -1/r  sum_{m>=1} Phi~_nl U_lm       F            (U_lm = P_lm / sin theta)
// acc = -grad Phi (not multiplied by the particle's mass); acc is ax[0..N) | ay | az.
// ---------------------------------------------------------------------------------------------
int oracle_scf_force(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                     double* acc, double* pot, int threads) {
    if (N < 1 || nmax < 0 || lmax < 0) return -1;
    const int L = num_lm(lmax);
    threads = resolve_threads(threads);
    const double *X = pos, *Y = pos + N, *Z = pos + 2 * N;
#pragma omp parallel num_threads(threads)
    {
        std::vector<double> P(L), dP(L), U(L), cm(lmax + 1), sm(lmax + 1);
        std::vector<double> Phi((nmax + 1) * (lmax + 1)), dPhi((nmax + 1) * (lmax + 1));
#pragma omp for schedule(static)
        for (long long k = 0; k < N; ++k) {
            Geom g = geometry(X[k], Y[k], Z[k]);
            legendre_table(lmax, g.ct, g.st, P.data(), dP.data(), U.data());
            trig_table(lmax, g.cp, g.sp, cm.data(), sm.data());
            radial_table(nmax, lmax, g.r, Phi.data(), dPhi.data());
            double sp = 0.0, sr = 0.0, st = 0.0, sf = 0.0;
            for (int n = 0; n <= nmax; ++n)
                for (int l = 0; l <= lmax; ++l)
                    for (int m = 0; m <= l; ++m) {
                        const int i = n * L + lm_index(l, m), j = lm_index(l, m), q = l * (nmax + 1) + n;
                        double E = A[i] * cm[m] + B[i] * sm[m];
                        double F = m * (-A[i] * sm[m] + B[i] * cm[m]);
                        sp += Phi[q] * P[j] * E;
                        sr += dPhi[q] * P[j] * E;
                        st += Phi[q] * dP[j] * E;
                        sf += Phi[q] * U[j] * F;
                    }
            double ar = -sr, at = -st / g.r, ap = -sf / g.r;
            to_cartesian(g, ar, at, ap, &acc[k], &acc[N + k], &acc[2 * N + k]);
            pot[k] = sp;
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// MEX sort ("sorted by r", "distance square ... for the sorting
// operation"; readings G7, G8): key = bits of r^2 with the pinned rounding
//   t = x*x;  t = fma(y,y,t);  t = fma(z,z,t)
// order = ascending (key, original index) = std::stable_sort on the key.  perm[rank] = index.
// ---------------------------------------------------------------------------------------------
int oracle_mex_sort(const double* pos, long long N, unsigned long long* keys, unsigned int* perm) {
    if (N < 1 || N >= (1LL << 31)) return -1;
    const double *X = pos, *Y = pos + N, *Z = pos + 2 * N;
    std::vector<uint64_t> key(N);
    for (long long k = 0; k < N; ++k) {
        double t = X[k] * X[k];
        t = std::fma(Y[k], Y[k], t);
        t = std::fma(Z[k], Z[k], t);
        std::memcpy(&key[k], &t, 8);
    }
    std::vector<uint32_t> idx(N);
    std::iota(idx.begin(), idx.end(), 0u);
    std::stable_sort(idx.begin(), idx.end(), [&](uint32_t a, uint32_t b) { return key[a] < key[b]; });
    for (long long k = 0; k < N; ++k) { perm[k] = idx[k]; if (keys) keys[k] = key[idx[k]]; }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// MEX force (eqs. 15–17 PAPER.md:146-155 with the discrete exclusive sums of eqs. 11–12
// PAPER.md:120-123).  With w_lm = (2-delta_m0)(l-m)!/(l+m)! and, for particle i (q, p held fixed:
// they are step functions of r):
//   q^{c,s}_lm(i) = sum_{rank(j)<rank(i)} m_j r_j^l      P_lm(j) {cos,sin}(m phi_j)
//   p^{c,s}_lm(i) = sum_{rank(j)>rank(i)} m_j r_j^-(l+1) P_lm(j) {cos,sin}(m phi_j)
//   Q^x = q^x r_i^-(l+1) + p^x r_i^l ;   R^x = -(l+1) q^x r_i^-(l+2) + l p^x r_i^(l-1)
//   Phi_i =        - sum w P_lm        (Q^c cos + Q^s sin)
//   a_r   =          sum w P_lm        (R^c cos + R^s sin)
//   a_th  =  1/r_i   sum w dP_lm/dth   (Q^c cos + Q^s sin)
//   a_phi =  1/r_i   sum_{m>=1} w U_lm m (-Q^c sin + Q^s cos)
// Streaming form: a forward sweep (inside-out) carries q and adds the q-part of (Phi, a); a backward
// sweep (outside-in) carries p and adds the p-part.  Particle i itself is excluded.
// perm_out (may be null) receives the sort permutation.
// ---------------------------------------------------------------------------------------------
int oracle_mex_force(const double* pos, const double* mass, long long N, int lmax,
                     double* acc, double* pot, unsigned int* perm_out) {
    if (N < 1 || N >= (1LL << 31) || lmax < 0) return -1;
    const int L = num_lm(lmax);
    const double *X = pos, *Y = pos + N, *Z = pos + 2 * N;
    std::vector<uint32_t> perm(N);
    oracle_mex_sort(pos, N, nullptr, perm.data());
    if (perm_out) std::memcpy(perm_out, perm.data(), sizeof(uint32_t) * N);

    std::vector<double> w(L);
    for (int l = 0; l <= lmax; ++l) for (int m = 0; m <= l; ++m) w[lm_index(l, m)] = w_lm(l, m);
    std::vector<double> P(L), dP(L), U(L), cm(lmax + 1), sm(lmax + 1);
    std::vector<double> sph(4 * (size_t)N, 0.0);   // Phi, a_r, a_th, a_phi per particle (by original index)

    for (int sweep = 0; sweep < 2; ++sweep) {      // 0: forward, carries q.  1: backward, carries p.
        std::vector<Neumaier> Mc(L), Ms(L);
        for (long long t = 0; t < N; ++t) {
            const long long rank = (sweep == 0) ? t : N - 1 - t;
            const uint32_t i = perm[rank];
            Geom g = geometry(X[i], Y[i], Z[i]);
            legendre_table(lmax, g.ct, g.st, P.data(), dP.data(), U.data());
            trig_table(lmax, g.cp, g.sp, cm.data(), sm.data());
            double sp = 0.0, sr = 0.0, st = 0.0, sf = 0.0;
            for (int l = 0; l <= lmax; ++l) {
                // radial factors of the evaluation (rq for the q-part, rp for the p-part) and of the moment
                double rad, drad, mom;
                if (sweep == 0) { rad = std::pow(g.r, -(l + 1)); drad = -(l + 1) * std::pow(g.r, -(l + 2)); mom = std::pow(g.r, l); }
                else { rad = std::pow(g.r, l); drad = (l == 0) ? 0.0 : l * std::pow(g.r, l - 1); mom = std::pow(g.r, -(l + 1)); }
                for (int m = 0; m <= l; ++m) {
                    const int j = lm_index(l, m);
                    const double Mcv = Mc[j].value(), Msv = Ms[j].value();
                    const double Qc = Mcv * rad, Qs = Msv * rad, Rc = Mcv * drad, Rs = Msv * drad;
                    sp += w[j] * P[j] * (Qc * cm[m] + Qs * sm[m]);
                    sr += w[j] * P[j] * (Rc * cm[m] + Rs * sm[m]);
                    st += w[j] * dP[j] * (Qc * cm[m] + Qs * sm[m]);
                    sf += w[j] * U[j] * m * (-Qc * sm[m] + Qs * cm[m]);
                    // now add particle i's own moment, AFTER it was evaluated (exclusive sums)
                    const double tmom = mass[i] * mom * P[j];
                    Mc[j].add(tmom * cm[m]);
                    Ms[j].add(tmom * sm[m]);
                }
            }
            sph[4 * (size_t)i + 0] += -sp;
            sph[4 * (size_t)i + 1] += sr;
            sph[4 * (size_t)i + 2] += st / g.r;
            sph[4 * (size_t)i + 3] += sf / g.r;
        }
    }
    for (long long i = 0; i < N; ++i) {
        Geom g = geometry(X[i], Y[i], Z[i]);
        pot[i] = sph[4 * (size_t)i];
        to_cartesian(g, sph[4 * (size_t)i + 1], sph[4 * (size_t)i + 2], sph[4 * (size_t)i + 3], &acc[i], &acc[N + i], &acc[2 * N + i]);
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// MEX force at a SAMPLE of particles, straight from the definition — no sort, no streaming carry.
// For sample particle i, eqs. (11)–(12) PAPER.md:120-123 are sums over "every j strictly interior"
// and "every j strictly exterior", where (readings G7, G8) j is interior to i iff
// (key_j, j) < (key_i, i) lexicographically, key = bits of r^2 with the pinned rounding.  So:
//   1. the S samples are ordered by (key, index);
//   2. every particle j (in index order, any order would do) is classified by b = number of samples
//      that are strictly interior to j (0..S).  j is exterior to samples[0..b), and interior to
//      samples[b'..S) with b' = b, or b + 1 when j is itself samples[b] (no self term);
//      its exterior-type moment m_j r_j^-(l+1) P_lm {cos,sin} is added to bin pbin[b], its
//      interior-type moment m_j r_j^l P_lm {cos,sin} to bin qbin[b'];
//   3. q(sample t) = sum_{b' <= t} qbin[b'],  p(sample t) = sum_{b > t} pbin[b];
//   4. Phi, a_r, a_theta, a_phi from the full expressions of the header comment above
//      (Q = q r^-(l+1) + p r^l, R = -(l+1) q r^-(l+2) + l p r^(l-1)), then spherical -> Cartesian.
// Used by the full-size GPU parity tests (N = 10^8), where the streaming sweep above would take
// minutes, and pinned against it at small N (tests/test_oracle_pins_mex.py).  OpenMP over j with
// thread-private bins combined in thread order; Neumaier sums throughout.
// acc_out is (3,S), pot_out (S), in the order of sample_idx.
// ---------------------------------------------------------------------------------------------
int oracle_mex_force_at(const double* pos, const double* mass, long long N, int lmax,
                        const long long* sample_idx, int S, double* acc_out, double* pot_out, int threads) {
    if (N < 1 || N >= (1LL << 31) || lmax < 0 || S < 1) return -1;
    const int L = num_lm(lmax);
    const double *X = pos, *Y = pos + N, *Z = pos + 2 * N;
    auto key_of = [&](long long k) {
        double t = X[k] * X[k];
        t = std::fma(Y[k], Y[k], t);
        t = std::fma(Z[k], Z[k], t);
        uint64_t u; std::memcpy(&u, &t, 8);
        return u;
    };
    for (int s = 0; s < S; ++s) if (sample_idx[s] < 0 || sample_idx[s] >= N) return -1;
    // 1. samples in (key, index) order; `where[t]` = position in sample_idx of the t-th sample
    std::vector<std::pair<uint64_t, long long>> so(S);
    std::vector<int> where(S);
    std::iota(where.begin(), where.end(), 0);
    std::sort(where.begin(), where.end(), [&](int a, int b) {
        return std::make_pair(key_of(sample_idx[a]), sample_idx[a]) < std::make_pair(key_of(sample_idx[b]), sample_idx[b]);
    });
    for (int t = 0; t < S; ++t) so[t] = std::make_pair(key_of(sample_idx[where[t]]), sample_idx[where[t]]);
    for (int t = 1; t < S; ++t) if (so[t] == so[t - 1]) return -2;   // duplicate sample indices

    threads = resolve_threads(threads);
    const size_t binsz = (size_t)(S + 1) * L;
    // per thread: qbin cos, qbin sin, pbin cos, pbin sin
    std::vector<std::vector<Neumaier>> bins(threads, std::vector<Neumaier>(4 * binsz));
#pragma omp parallel num_threads(threads)
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num();
#else
        const int tid = 0;
#endif
        Neumaier* qc = bins[tid].data();
        Neumaier* qs = qc + binsz;
        Neumaier* pc = qs + binsz;
        Neumaier* ps = pc + binsz;
        std::vector<double> P(L), dP(L), U(L), cm(lmax + 1), sm(lmax + 1);
#pragma omp for schedule(static)
        for (long long j = 0; j < N; ++j) {
            const std::pair<uint64_t, long long> me(key_of(j), j);
            const int b = (int)(std::lower_bound(so.begin(), so.end(), me) - so.begin());   // samples strictly interior to j
            const int bq = (b < S && so[b] == me) ? b + 1 : b;
            Geom g = geometry(X[j], Y[j], Z[j]);
            legendre_table(lmax, g.ct, g.st, P.data(), dP.data(), U.data());
            trig_table(lmax, g.cp, g.sp, cm.data(), sm.data());
            for (int l = 0; l <= lmax; ++l) {
                const double mq = mass[j] * std::pow(g.r, l), mp = mass[j] * std::pow(g.r, -(l + 1));
                for (int m = 0; m <= l; ++m) {
                    const int i = lm_index(l, m);
                    if (bq <= S - 1) { qc[(size_t)bq * L + i].add(mq * P[i] * cm[m]); qs[(size_t)bq * L + i].add(mq * P[i] * sm[m]); }
                    if (b >= 1) { pc[(size_t)b * L + i].add(mp * P[i] * cm[m]); ps[(size_t)b * L + i].add(mp * P[i] * sm[m]); }
                }
            }
        }
    }
    // combine threads in thread order
    std::vector<Neumaier> tot(4 * binsz);
    for (int t = 0; t < threads; ++t)
        for (size_t i = 0; i < 4 * binsz; ++i) { tot[i].add(bins[t][i].s); tot[i].add(bins[t][i].c); }
    const Neumaier *qc = tot.data(), *qs = qc + binsz, *pc = qs + binsz, *ps = pc + binsz;

    std::vector<double> P(L), dP(L), U(L), cm(lmax + 1), sm(lmax + 1);
    for (int t = 0; t < S; ++t) {
        // 3. exclusive sums of sample t
        std::vector<Neumaier> Qc(L), Qs(L), Pc(L), Ps(L);
        for (int b = 0; b <= t; ++b) for (int i = 0; i < L; ++i) { Qc[i].add(qc[(size_t)b * L + i].value()); Qs[i].add(qs[(size_t)b * L + i].value()); }
        for (int b = S; b > t; --b) for (int i = 0; i < L; ++i) { Pc[i].add(pc[(size_t)b * L + i].value()); Ps[i].add(ps[(size_t)b * L + i].value()); }
        // 4. evaluate
        const long long k = so[t].second;
        Geom g = geometry(X[k], Y[k], Z[k]);
        legendre_table(lmax, g.ct, g.st, P.data(), dP.data(), U.data());
        trig_table(lmax, g.cp, g.sp, cm.data(), sm.data());
        double sp = 0.0, sr = 0.0, st = 0.0, sf = 0.0;
        for (int l = 0; l <= lmax; ++l) {
            const double ri = std::pow(g.r, -(l + 1)), rl = std::pow(g.r, l);
            const double dri = -(l + 1) * std::pow(g.r, -(l + 2)), drl = (l == 0) ? 0.0 : l * std::pow(g.r, l - 1);
            for (int m = 0; m <= l; ++m) {
                const int i = lm_index(l, m);
                const double w = w_lm(l, m);
                const double Qcv = Qc[i].value() * ri + Pc[i].value() * rl, Qsv = Qs[i].value() * ri + Ps[i].value() * rl;
                const double Rcv = Qc[i].value() * dri + Pc[i].value() * drl, Rsv = Qs[i].value() * dri + Ps[i].value() * drl;
                sp += w * P[i] * (Qcv * cm[m] + Qsv * sm[m]);
                sr += w * P[i] * (Rcv * cm[m] + Rsv * sm[m]);
                st += w * dP[i] * (Qcv * cm[m] + Qsv * sm[m]);
                sf += w * U[i] * m * (-Qcv * sm[m] + Qsv * cm[m]);
            }
        }
        const int o = where[t];
        pot_out[o] = -sp;
        to_cartesian(g, sr, st / g.r, sf / g.r, &acc_out[o], &acc_out[S + o], &acc_out[2 * S + o]);
    }
    return 0;
}

}  // extern "C"

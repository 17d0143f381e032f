// etics_common.cuh — shared by the CUDA translation units of libetics (never by oracle/).
//
// Holds: limits, the (l,m) index map, the basis-constant tables (host generator + __constant__ copy per
// translation unit), per-particle geometry, and small launch helpers.  Formulas: DESIGN.md "Readings" G1
// (HO92 basis, cited by PAPER.md:183 §2.5 but not printed there) and SURVEY.md §8(c).
#pragma once

#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <mutex>

#include "../../include/etics.h"

namespace etics {

constexpr int kMaxL = ETICS_MAX_LMAX;
constexpr int kMaxN = ETICS_MAX_NMAX;
constexpr int kMaxLM = (kMaxL + 1) * (kMaxL + 2) / 2;

__host__ __device__ constexpr int lm_index(int l, int m) { return l * (l + 1) / 2 + m; }
__host__ __device__ constexpr int num_lm(int lmax) { return (lmax + 1) * (lmax + 2) / 2; }

// ---------------------------------------------------------------------------------------------------------
// Basis constants.
//   Gegenbauer recurrence for alpha = 2l + 3/2 (the paper's W_nl), written with reciprocal-free
//   coefficients:  C_n = a_n xi C_{n-1} - b_n C_{n-2},  a_n = 2(n+alpha-1)/n,  b_n = (n+2alpha-2)/n,  C_{-1}=0, C_0=1.
//   A~_nl = 4 pi / I_nl,  I_nl = -K_nl 4 pi g(n,l) / (n + 2l + 3/2),  K_nl = n(n+4l+3)/2 + (l+1)(2l+1),
//   g(n,l) = Gamma(n+4l+3) / (n! Gamma(2l+3/2)^2 2^(8l+6)) built by exact ratio recurrences:
//     g(0,0) = 1/(8 pi);  g(0,l+1)/g(0,l) = (4l+3)(4l+4)(4l+5)(4l+6) / (256 (2l+3/2)^2 (2l+5/2)^2);
//     g(n+1,l)/g(n,l) = (n+4l+3)/(n+1).
//   N_lm = (2-delta_m0)(2l+1)/(4 pi) (l-m)!/(l+m)!   (SCF: +-m folded into m >= 0),
//   w_lm = (2-delta_m0)(l-m)!/(l+m)!                 (MEX weight, = N_lm 4 pi/(2l+1)).
// ---------------------------------------------------------------------------------------------------------
struct BasisConstants {
    double geg_a[kMaxL + 1][kMaxN + 2];
    double geg_b[kMaxL + 1][kMaxN + 2];
    // monic forms used by the coefficient accumulation (scales are folded into the final normalisation):
    //   C_n = g_n Q_n,  Q_n = xi Q_{n-1} - beta_n Q_{n-2},  g_n = prod a_i,  beta_n = b_n / (a_n a_{n-1})
    //   P_lm = h_lm q_l, q_m = st^m, q_l = ct q_{l-1} - gamma_lm q_{l-2},  h_mm = (2m-1)!!, h_lm = h_{l-1,m} (2l-1)/(l-m)
    double geg_beta[kMaxL + 1][kMaxN + 2];
    double geg_scale[kMaxL + 1][kMaxN + 1];
    double leg_gamma_T[kMaxL + 1][kMaxL + 2];   // [m][l], zero for l < m+2 (and the slack entry l = kMaxL+1)
    double leg_scale[kMaxL + 1][kMaxL + 1];   // [l][m]
    double norm_nl[kMaxL + 1][kMaxN + 1];   // A~_nl
    double N_lm[kMaxLM];
    double w_lm[kMaxLM];
};

inline void fill_basis_constants(BasisConstants& c) {
    const long double pi = 3.14159265358979323846264338327950288L;
    long double g0 = 1.0L / (8.0L * pi);
    for (int l = 0; l <= kMaxL; ++l) {
        const long double alpha = 2.0L * l + 1.5L;
        c.geg_a[l][0] = 0.0; c.geg_b[l][0] = 0.0;
        for (int n = 1; n <= kMaxN + 1; ++n) {
            c.geg_a[l][n] = (double)(2.0L * (n + alpha - 1.0L) / n);
            c.geg_b[l][n] = (double)((n + 2.0L * alpha - 2.0L) / n);
        }
        long double g = g0;
        for (int n = 0; n <= kMaxN; ++n) {
            const long double K = 0.5L * n * (n + 4.0L * l + 3.0L) + (l + 1.0L) * (2.0L * l + 1.0L);
            const long double I = -K * 4.0L * pi * g / (n + 2.0L * l + 1.5L);
            c.norm_nl[l][n] = (double)(4.0L * pi / I);
            g = g * (n + 4.0L * l + 3.0L) / (n + 1.0L);
        }
        const long double h1 = 2.0L * l + 1.5L, h2 = 2.0L * l + 2.5L;
        g0 = g0 * (4.0L * l + 3.0L) * (4.0L * l + 4.0L) * (4.0L * l + 5.0L) * (4.0L * l + 6.0L) / (256.0L * h1 * h1 * h2 * h2);
    }
    for (int l = 0; l <= kMaxL; ++l) {
        const long double alpha = 2.0L * l + 1.5L;
        long double g = 1.0L, aprev = 1.0L;
        c.geg_beta[l][0] = 0.0; c.geg_beta[l][1] = 0.0; c.geg_scale[l][0] = 1.0;
        for (int n = 1; n <= kMaxN + 1; ++n) {
            const long double a = 2.0L * (n + alpha - 1.0L) / n, b = (n + 2.0L * alpha - 2.0L) / n;
            if (n >= 2) c.geg_beta[l][n] = (double)(b / (a * aprev));
            g *= a;
            if (n <= kMaxN) c.geg_scale[l][n] = (double)g;
            aprev = a;
        }
    }
    for (int m = 0; m <= kMaxL; ++m) {
        long double h = 1.0L, aprev = 1.0L;
        for (int k = 1; k <= m; ++k) h *= (2.0L * k - 1.0L);
        for (int l = 0; l <= kMaxL + 1; ++l) c.leg_gamma_T[m][l] = 0.0;
        for (int l = 0; l <= kMaxL; ++l) c.leg_scale[l][m] = 0.0;
        c.leg_scale[m][m] = (double)h;
        for (int l = m + 1; l <= kMaxL; ++l) {
            const long double a = (2.0L * l - 1.0L) / (l - m), b = (l + m - 1.0L) / (l - m);
            if (l >= m + 2) c.leg_gamma_T[m][l] = (double)(b / (a * aprev));
            h *= a;
            c.leg_scale[l][m] = (double)h;
            aprev = a;
        }
    }
    for (int l = 0; l <= kMaxL; ++l)
        for (int m = 0; m <= l; ++m) {
            long double f = 1.0L;
            for (int k = l - m + 1; k <= l + m; ++k) f /= k;
            const long double w = (m == 0 ? 1.0L : 2.0L) * f;
            c.w_lm[lm_index(l, m)] = (double)w;
            c.N_lm[lm_index(l, m)] = (double)(w * (2 * l + 1) / (4.0L * pi));
        }
}

// One-time set-up per DEVICE (function attributes and __constant__ copies belong to a device; one process may
// drive several GPUs, and several host threads may call in): run(f) calls f once for the current device.
struct DeviceOnce {
    std::mutex mu;
    std::atomic<bool> done[64] = {};
    template <class F>
    cudaError_t run(F&& f) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        if (dev < 0 || dev >= 64) return f();
        if (done[dev].load(std::memory_order_acquire)) return cudaSuccess;
        std::lock_guard<std::mutex> lock(mu);
        if (done[dev].load(std::memory_order_relaxed)) return cudaSuccess;
        e = f();
        if (e == cudaSuccess) done[dev].store(true, std::memory_order_release);
        return e;
    }
};

// SM count of the current device (148 when no device is present, so that size queries work on a CPU-only box).
inline int device_sm_count() {
    static std::atomic<int> sms[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    int v = sms[dev].load(std::memory_order_relaxed);
    if (v == 0) {
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
        sms[dev].store(v, std::memory_order_relaxed);
    }
    return v;
}

// One __constant__ copy per translation unit (no relocatable device code needed); uploaded by the unit's per-device init.
#define ETICS_DEFINE_CONSTANTS()                                                                     \
    static __constant__ etics::BasisConstants c_basis;                                               \
    static cudaError_t etics_upload_constants_now() {                                                \
        etics::BasisConstants* host = new etics::BasisConstants;                                     \
        etics::fill_basis_constants(*host);                                                          \
        cudaError_t e = cudaMemcpyToSymbol(c_basis, host, sizeof(*host));                            \
        delete host;                                                                                 \
        return e;                                                                                    \
    }

// ---------------------------------------------------------------------------------------------------------
// Per-particle geometry.  On-axis particles: phi := 0.
// ---------------------------------------------------------------------------------------------------------
struct Geom { double r, rinv, ct, st, cp, sp; };

__device__ __forceinline__ Geom geometry(double x, double y, double z) {
    // reciprocal square roots (MUFU.RSQ64H + Newton, <= 1 ulp) instead of sqrt + divide: 1/r and 1/rho are what
    // the path needs, r = r^2 (1/r) and rho = rho^2 (1/rho) follow with one multiply each
    Geom g;
    const double rho2 = fma(y, y, x * x);
    const double r2 = fma(z, z, rho2);
    g.rinv = rsqrt(r2);
    g.r = r2 * g.rinv;
    g.ct = z * g.rinv;
    if (rho2 > 0.0) {
        const double ri = rsqrt(rho2);
        g.st = (rho2 * ri) * g.rinv;
        g.cp = x * ri;
        g.sp = y * ri;
    } else {
        g.st = 0.0;
        g.cp = 1.0;
        g.sp = 0.0;
    }
    return g;
}

// Spherical -> Cartesian (the paper's last kernel, fused here).
__device__ __forceinline__ void to_cartesian(const Geom& g, double ar, double at, double ap,
                                             double& ax, double& ay, double& az) {
    const double h = fma(ar, g.st, at * g.ct);   // component along the cylindrical radius
    ax = fma(h, g.cp, -ap * g.sp);
    ay = fma(h, g.sp, ap * g.cp);
    az = fma(ar, g.ct, -at * g.st);
}

inline size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Internal launchers (one per translation unit), called by the C ABI in etics_api.cu.
cudaError_t scf_init_constants();
size_t scf_coeffs_workspace(long long N, int nmax, int lmax);
cudaError_t scf_coeffs_launch(const double* pos, const double* mass, long long N, int nmax, int lmax,
                              double* A, double* B, void* ws, cudaStream_t st);
int scf_coeffs_blocks(long long N, int nmax, int lmax, long long* particles_per_block);
cudaError_t scf_accumulate_launch(const double* pos, const double* mass, long long N, int nmax, int lmax, void* ws,
                                  int block0, int nblocks, cudaStream_t st);
cudaError_t scf_finalize_launch(long long N, int nmax, int lmax, double* A, double* B, const void* ws, cudaStream_t st);
cudaError_t scf_force_launch(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B, int what,
                             double* acc, double* pot, cudaStream_t st);

size_t scf_force_f32_workspace(int nmax, int lmax);
cudaError_t scf_force_f32_launch(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                                 double* acc, double* pot, void* ws, cudaStream_t st);
cudaError_t scf_combine_launch(const double* parts, int nparts, long long len, double* out, cudaStream_t st);

cudaError_t mex_init_constants();
int mex_kernel_launches(long long N);
size_t mex_workspace(long long N, int lmax);
cudaError_t mex_sort_launch(const double* pos, long long N, unsigned long long* keys_sorted, unsigned int* perm,
                            void* ws, cudaStream_t st);
cudaError_t mex_force_launch(const double* pos, const double* mass, long long N, int lmax, int what,
                             double* acc, double* pot, void* ws, cudaStream_t st);

cudaError_t mex_force_timed(const double* pos, const double* mass, long long N, int lmax, double* acc, double* pot,
                            void* ws, cudaStream_t st, float* stage_ms);
// radius-partitioned MEX: the force sequence cut at the exchange of the shards' moment vectors
int mex_shard_rows(int lmax);
cudaError_t mex_shard_moments_launch(const double* pos, const double* mass, long long N, int lmax, double* totals, void* ws,
                                     cudaStream_t st);
cudaError_t mex_shard_bases_launch(const double* parts, int nparts, int rank, int lmax, double* base, cudaStream_t st);
cudaError_t mex_shard_force_launch(long long N, int lmax, int what, const double* base, double* acc, double* pot, void* ws,
                                   cudaStream_t st);

cudaError_t probe_dfma_launch(int iters, double* sink, double* flops_out, cudaStream_t st);
cudaError_t probe_copy_launch(void* dst, const void* src, size_t bytes, cudaStream_t st);

}  // namespace etics

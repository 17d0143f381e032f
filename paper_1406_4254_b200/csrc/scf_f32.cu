// scf_f32.cu — single-precision SCF evaluation (§3.4: "the single-precision ... speed-up",
// PAPER.md:331-354 §4.2: the single-precision study and its failure near the z axis).
//
// Same sums as scf_eval_kernel (scf.cu), every per-particle quantity in fp32: geometry, the monic Legendre l-recurrence at
// fixed m, the Gegenbauer recurrence and its derivative, the sums over n and (l, m), the transform to Cartesian.  Inputs
// (pos, A, B) and outputs (acc, pot) stay fp64 arrays: the coefficients come from the fp64 accumulation over particles
// (that sum over N terms is where single precision costs most), only the O(T) work per particle drops to fp32.
// The paper's fp32 runs lose all accuracy near the z axis because eq. 24 recurs upward in m from P_l0, P_l1
// (PAPER.md:344-350).  Nothing of that kind happens here: the l-recurrence at fixed m starts from sin^m(theta) and
// U_lm = P_lm / sin(theta) is a polynomial of its own, so nothing is divided by sin(theta) and no cancelling pair is formed
// (tests/test_gpu_scf.py::test_f32_mode_is_accurate_near_the_z_axis).
#include "etics_common.cuh"

namespace etics {

struct BasisConstantsF32 {
    float geg_a[kMaxL + 1][kMaxN + 2];
    float geg_b[kMaxL + 1][kMaxN + 2];
    double leg_scale[kMaxL + 1][kMaxL + 1];   // h_lm of the monic Legendre rows (fp64: the table entries are rounded once)
};
static __constant__ BasisConstantsF32 c_f32;

__host__ __device__ constexpr float leg_gamma_f(int l, int m) {
    return (l >= m + 2) ? float(double((l + m - 1) * (l - 1 - m)) / double((2 * l - 1) * (2 * l - 3))) : 0.0f;
}

constexpr int kF32Threads = 256;

template <int LMAX>
__global__ void __launch_bounds__(kF32Threads, 2)
scf_eval_f32_kernel(const double* __restrict__ pos, long long N, int nmax, const float2* __restrict__ tab,
                    double* __restrict__ acc, double* __restrict__ pot) {
    extern __shared__ float2 s_tab[];   // (A, B) h_lm pairs, index n1*l(l+1)/2 + n*(l+1) + m, packed by scf_pack_f32_kernel
    constexpr int L = num_lm(LMAX);
    const int n1 = nmax + 1;
    for (int g = threadIdx.x; g < n1 * L; g += kF32Threads) s_tab[g] = tab[g];
    __syncthreads();
    const long long k = (long long)blockIdx.x * kF32Threads + threadIdx.x;
    if (k >= N) return;

    // ---- geometry (S1), fp32 ----------------------------------------------------------------------------------
    const float x = (float)pos[k], y = (float)pos[N + k], z = (float)pos[2 * N + k];
    const float rho2 = fmaf(y, y, x * x), r2 = fmaf(z, z, rho2);
    const float rinv = rsqrtf(r2), r = r2 * rinv, ct = z * rinv;
    float st = 0.0f, cp = 1.0f, sp = 0.0f;
    if (rho2 > 0.0f) {
        const float ri = rsqrtf(rho2);
        st = (rho2 * ri) * rinv; cp = x * ri; sp = y * ri;
    }
    float cm[LMAX + 1], sm[LMAX + 1];
    cm[0] = 1.0f; sm[0] = 0.0f;
#pragma unroll
    for (int m = 1; m <= LMAX; ++m) {
        cm[m] = fmaf(cm[m - 1], cp, -sm[m - 1] * sp);
        sm[m] = fmaf(sm[m - 1], cp, cm[m - 1] * sp);
    }
    const float u = __frcp_rn(1.0f + r);
    const float xi = (r - 1.0f) * u, s = r * u * u, xr = xi * rinv, two_u2 = 2.0f * u * u;
    float fl = -u, gl = -u;
    float s_pot = 0.0f, s_r = 0.0f, s_t = 0.0f, s_f = 0.0f;
    float U1[LMAX + 1], U2[LMAX + 1];   // rows l-1 and l-2 of (P_l0, U_l1, ..., U_ll), monic
    const float2* tl = s_tab;

#pragma unroll
    for (int l = 0; l <= LMAX; ++l) {
        float U0[LMAX + 1];
        if (l == 0) {
            U0[0] = 1.0f;
        } else if (l == 1) {
            U0[0] = ct; U0[1] = 1.0f;
        } else {
#pragma unroll
            for (int m = 0; m <= l - 2; ++m) U0[m] = fmaf(ct, U1[m], -leg_gamma_f(l, m) * U2[m]);
            U0[l - 1] = ct * U1[l - 1];
            U0[l] = st * U1[l - 1];
        }
        float sa[LMAX + 1], sad[LMAX + 1], sb[LMAX + 1], sbd[LMAX + 1];
#pragma unroll
        for (int m = 0; m <= l; ++m) { sa[m] = 0.0f; sad[m] = 0.0f; sb[m] = 0.0f; sbd[m] = 0.0f; }
        float C = 1.0f, Cm = 0.0f, D = 0.0f, Dm = 0.0f;   // C_n, C_{n-1}, dC_n/dxi, dC_{n-1}/dxi
#pragma unroll 2
        for (int n = 0; n < n1; ++n) {
#pragma unroll
            for (int m = 0; m <= l; ++m) {
                const float2 ab = tl[n * (l + 1) + m];
                sa[m] = fmaf(ab.x, C, sa[m]);
                sad[m] = fmaf(ab.x, D, sad[m]);
                if (m > 0) {
                    sb[m] = fmaf(ab.y, C, sb[m]);
                    sbd[m] = fmaf(ab.y, D, sbd[m]);
                }
            }
            const float a = c_f32.geg_a[l][n + 1], b = c_f32.geg_b[l][n + 1];
            const float ax = a * xi;
            const float Cn = fmaf(ax, C, -b * Cm);
            const float Dn = fmaf(ax, D, fmaf(a, C, -b * Dm));
            Cm = C; C = Cn; Dm = D; D = Dn;
        }
        tl += n1 * (l + 1);

        float lv_p = 0.0f, lv_r = 0.0f, lv_t = 0.0f, lv_f = 0.0f;
        const float lct = float(l) * ct;
#pragma unroll
        for (int m = 0; m <= l; ++m) {
            const float Ea = (m == 0) ? sa[0] : fmaf(sa[m], cm[m], sb[m] * sm[m]);
            const float Ed = (m == 0) ? sad[0] : fmaf(sad[m], cm[m], sbd[m] * sm[m]);
            float P, dP;
            if (m == 0) {
                P = U0[0];
                dP = (l >= 1) ? -(float(l) * st) * U0[1] : 0.0f;
            } else {
                P = st * U0[m];
                dP = (m < l) ? fmaf(lct, U0[m], -float(double((l + m) * (l - m)) / double(2 * l - 1)) * U1[m]) : lct * U0[m];
            }
            lv_p = fmaf(P, Ea, lv_p);
            lv_r = fmaf(P, Ed, lv_r);
            lv_t = fmaf(dP, Ea, lv_t);
            if (m > 0) lv_f = fmaf(float(m) * U0[m], fmaf(sb[m], cm[m], -sa[m] * sm[m]), lv_f);
        }
        s_pot = fmaf(fl, lv_p, s_pot);
        s_r = fmaf(fl, fmaf(gl, lv_p, two_u2 * lv_r), s_r);
        s_t = fmaf(fl, lv_t, s_t);
        s_f = fmaf(fl, lv_f, s_f);
        fl *= s;
        gl -= xr;
#pragma unroll
        for (int m = 0; m <= l; ++m) { U2[m] = U1[m]; U1[m] = U0[m]; }
    }
    if (acc) {
        const float ar = -s_r, at = -s_t * rinv, ap = -s_f * rinv;
        const float h = fmaf(ar, st, at * ct);
        acc[k] = (double)fmaf(h, cp, -ap * sp);
        acc[N + k] = (double)fmaf(h, sp, ap * cp);
        acc[2 * N + k] = (double)fmaf(ar, ct, -at * st);
    }
    if (pot) pot[k] = (double)s_pot;
}

// (A, B) fp64 -> the evaluation table in fp32, scaled by the Legendre scale h_lm of the monic rows (the products are formed
// in fp64 and rounded once).
__global__ void __launch_bounds__(256)
scf_pack_f32_kernel(const double* __restrict__ A, const double* __restrict__ B, int nmax, int lmax, float2* __restrict__ tab) {
    const int L = num_lm(lmax), n1 = nmax + 1;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n1 * L) return;
    const int n = g / L, j = g - n * L;
    int l = 0;
    while (lm_index(l + 1, 0) <= j) ++l;
    const int m = j - lm_index(l, 0);
    const double sc = c_f32.leg_scale[l][m];
    tab[n1 * lm_index(l, 0) + n * (l + 1) + m] = make_float2((float)(A[g] * sc), (float)(B[g] * sc));
}

static cudaError_t f32_init() {
    static DeviceOnce once;
    return once.run([] {
        BasisConstants* full = new BasisConstants;
        fill_basis_constants(*full);
        BasisConstantsF32* h = new BasisConstantsF32;
        for (int l = 0; l <= kMaxL; ++l)
            for (int n = 0; n < kMaxN + 2; ++n) { h->geg_a[l][n] = (float)full->geg_a[l][n]; h->geg_b[l][n] = (float)full->geg_b[l][n]; }
        for (int l = 0; l <= kMaxL; ++l)
            for (int m = 0; m <= kMaxL; ++m) h->leg_scale[l][m] = full->leg_scale[l][m];
        cudaError_t e = cudaMemcpyToSymbol(c_f32, h, sizeof(*h));
        delete h;
        delete full;
        return e;
    });
}

size_t scf_force_f32_workspace(int nmax, int lmax) {
    return round_up((size_t)(nmax + 1) * num_lm(lmax) * sizeof(float2), 256);
}

template <int LMAX>
static cudaError_t launch_f32(const double* pos, long long N, int nmax, const float2* tab, double* acc, double* pot, cudaStream_t st) {
    const size_t smem = (size_t)(nmax + 1) * num_lm(LMAX) * sizeof(float2);
    scf_eval_f32_kernel<LMAX><<<(unsigned)((N + kF32Threads - 1) / kF32Threads), kF32Threads, smem, st>>>(pos, N, nmax, tab, acc, pot);
    return cudaGetLastError();
}

// workspace: the packed fp32 table
cudaError_t scf_force_f32_launch(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                                 double* acc, double* pot, void* ws, cudaStream_t st) {
    cudaError_t e = f32_init();
    if (e != cudaSuccess) return e;
    float2* tab = static_cast<float2*>(ws);
    const int T = (nmax + 1) * num_lm(lmax);
    scf_pack_f32_kernel<<<(T + 255) / 256, 256, 0, st>>>(A, B, nmax, lmax, tab);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    switch (lmax) {
#define ETICS_CASE(LM) case LM: return launch_f32<LM>(pos, N, nmax, tab, acc, pot, st);
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5)
        ETICS_CASE(6) ETICS_CASE(7) ETICS_CASE(8) ETICS_CASE(9) ETICS_CASE(10)
#undef ETICS_CASE
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace etics

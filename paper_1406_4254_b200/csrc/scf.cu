// scf.cu — SCF half of the hot path (SURVEY.md §8(a) S1–S7) for sm_100a.
//
//   scf_accumulate_kernel  S1–S4: per-particle geometry, Legendre/trig and Gegenbauer recurrences in registers,
//                          features staged once through shared memory, register-tiled accumulation of
//                          S^{c,s}_nlm, one partial table per block in a fixed particle order.
//   scf_finalize_kernel    S5: fixed-order reduction over the block partials, times A~_nl N_lm -> A, B.
//   scf_eval_kernel        S6–S7: (A,B) table broadcast from shared memory, per-particle recurrences with
//                          derivatives, sums over n then (l,m) in registers, spherical -> Cartesian, store.
//
// What the paper did instead (prior art, §3.3): one kernel launch per (n,l) pair with a
// shared-memory block reduction, block partials copied to the host and summed by the CPU, coefficients copied
// back into constant memory, then one force kernel plus a separate coordinate-transform kernel.
// No fp64 atomics anywhere: results are bitwise reproducible run to run.
#include "etics_common.cuh"

namespace etics {

ETICS_DEFINE_CONSTANTS()

cudaError_t scf_init_constants() { return etics_upload_constants(); }

// =========================================================================================================
// Evaluation kernel (S6–S7).  One thread per particle; template on lmax so that every (l,m) array lives in
// registers; the n loop is a runtime loop.  Loop order l -> n -> m as in PAPER.md:251.
//
// Per level l (alpha = 2l+3/2, xi = (r-1)/(r+1), u = 1/(1+r), s = r u^2):
//   Phi~_nl = f_l C_n(xi),  f_l = -u s^l;   dPhi~_nl/dr = f_l ( g_l C_n + 2 u^2 C'_n ),  g_l = f_l'/f_l = -u - l xi / r
//   SA_m = sum_n A_nlm C_n, SAd_m = sum_n A_nlm C'_n (SB, SBd likewise)  -> 4 FMA per (n,l,m), operand from smem
//   E_m = SA_m cos(m phi) + SB_m sin(m phi), Ed_m likewise with SAd/SBd, F_m = SB_m cos - SA_m sin
//   Phi   += f_l sum_m P_lm E_m
//   dPhi/dr    += f_l ( g_l sum_m P_lm E_m + 2u^2 sum_m P_lm Ed_m )
//   dPhi/dth   += f_l sum_m dP_lm E_m
//   (1/sin th) dPhi/dphi += f_l sum_m m U_lm F_m,   U_lm = P_lm / sin(theta) from its own recurrence
// =========================================================================================================
constexpr int kEvalThreads = 128;

template <int LMAX>
__global__ void __launch_bounds__(kEvalThreads)
scf_eval_kernel(const double* __restrict__ pos, long long N, int nmax,
                const double* __restrict__ A, const double* __restrict__ B,
                double* __restrict__ acc, double* __restrict__ pot) {
    extern __shared__ double2 s_tab[];   // (A,B) pairs, index n1*l(l+1)/2 + n*(l+1) + m
    constexpr int L = num_lm(LMAX);
    const int n1 = nmax + 1;
    for (int g = threadIdx.x; g < n1 * L; g += kEvalThreads) {
        const int n = g / L, j = g - n * L;
        int l = 0;
        while (lm_index(l + 1, 0) <= j) ++l;
        const int m = j - lm_index(l, 0);
        s_tab[n1 * lm_index(l, 0) + n * (l + 1) + m] = make_double2(A[g], B[g]);
    }
    __syncthreads();

    const long long k = (long long)blockIdx.x * kEvalThreads + threadIdx.x;
    if (k >= N) return;
    const Geom g = geometry(pos[k], pos[N + k], pos[2 * N + k]);

    double cm[LMAX + 1], sm[LMAX + 1];
    cm[0] = 1.0; sm[0] = 0.0;
#pragma unroll
    for (int m = 1; m <= LMAX; ++m) {
        cm[m] = fma(cm[m - 1], g.cp, -sm[m - 1] * g.sp);
        sm[m] = fma(sm[m - 1], g.cp, cm[m - 1] * g.sp);
    }

    const double u = 1.0 / (1.0 + g.r);
    const double xi = (g.r - 1.0) * u;
    const double s = g.r * u * u;
    const double xr = xi * g.rinv;
    const double two_u2 = 2.0 * u * u;
    double fl = -u, gl = -u;
    double s_pot = 0.0, s_r = 0.0, s_t = 0.0, s_f = 0.0;
    double U1[LMAX + 1], U2[LMAX + 1];   // rows l-1 and l-2 of (P_l0, U_l1, ..., U_ll)
    const double2* tl = s_tab;

#pragma unroll
    for (int l = 0; l <= LMAX; ++l) {
        // ---- angular row l (stable l-recurrence; no division by sin theta) ------------------------------
        double U0[LMAX + 1];
        if (l == 0) {
            U0[0] = 1.0;
        } else if (l == 1) {
            U0[0] = g.ct; U0[1] = 1.0;
        } else {
#pragma unroll
            for (int m = 0; m <= l - 2; ++m) {
                const double a = double(2 * l - 1) / double(l - m), b = double(l + m - 1) / double(l - m);
                U0[m] = fma(a * g.ct, U1[m], -b * U2[m]);
            }
            U0[l - 1] = double(2 * l - 1) * g.ct * U1[l - 1];
            U0[l] = double(2 * l - 1) * g.st * U1[l - 1];
        }
        double Pm[LMAX + 2];
        Pm[0] = U0[0];
#pragma unroll
        for (int m = 1; m <= l; ++m) Pm[m] = g.st * U0[m];
        Pm[l + 1] = 0.0;

        // ---- radial sums over n -----------------------------------------------------------------------
        double sa[LMAX + 1], sad[LMAX + 1], sb[LMAX + 1], sbd[LMAX + 1];
#pragma unroll
        for (int m = 0; m <= l; ++m) { sa[m] = 0.0; sad[m] = 0.0; sb[m] = 0.0; sbd[m] = 0.0; }
        double C = 1.0, Cm = 0.0, D = 0.0, Dm = 0.0;
        for (int n = 0; n < n1; ++n) {
#pragma unroll
            for (int m = 0; m <= l; ++m) {
                const double2 ab = tl[n * (l + 1) + m];
                sa[m] = fma(ab.x, C, sa[m]);
                sad[m] = fma(ab.x, D, sad[m]);
                if (m > 0) {
                    sb[m] = fma(ab.y, C, sb[m]);
                    sbd[m] = fma(ab.y, D, sbd[m]);
                }
            }
            const double a = c_basis.geg_a[l][n + 1], b = c_basis.geg_b[l][n + 1];
            const double ax = a * xi;
            const double Cn = fma(ax, C, -b * Cm);
            const double Dn = fma(ax, D, fma(a, C, -b * Dm));
            Cm = C; C = Cn; Dm = D; D = Dn;
        }
        tl += n1 * (l + 1);

        // ---- combine the level ------------------------------------------------------------------------
        double lv_p = 0.0, lv_r = 0.0, lv_t = 0.0, lv_f = 0.0;
#pragma unroll
        for (int m = 0; m <= l; ++m) {
            const double Ea = fma(sa[m], cm[m], sb[m] * sm[m]);
            const double Ed = fma(sad[m], cm[m], sbd[m] * sm[m]);
            double dP;
            if (m == 0) dP = -Pm[1];
            else dP = fma(0.5 * double((l + m) * (l - m + 1)), Pm[m - 1], -0.5 * Pm[m + 1]);
            lv_p = fma(Pm[m], Ea, lv_p);
            lv_r = fma(Pm[m], Ed, lv_r);
            lv_t = fma(dP, Ea, lv_t);
            if (m > 0) {
                const double Fa = fma(sb[m], cm[m], -sa[m] * sm[m]);
                lv_f = fma(double(m) * U0[m], Fa, lv_f);
            }
        }
        s_pot = fma(fl, lv_p, s_pot);
        s_r = fma(fl, fma(gl, lv_p, two_u2 * lv_r), s_r);
        s_t = fma(fl, lv_t, s_t);
        s_f = fma(fl, lv_f, s_f);
        fl *= s;
        gl -= xr;
#pragma unroll
        for (int m = 0; m <= l; ++m) { U2[m] = U1[m]; U1[m] = U0[m]; }
    }

    double ax, ay, az;
    to_cartesian(g, -s_r, -s_t * g.rinv, -s_f * g.rinv, ax, ay, az);
    acc[k] = ax;
    acc[N + k] = ay;
    acc[2 * N + k] = az;
    pot[k] = s_pot;
}

// =========================================================================================================
// Coefficient accumulation (S1–S4).
//
// The sum S_l[n][y] = sum_k R_l[k][n] Y_l[k][y] (R = m_k Phi~_nl, Y = P_lm {cos,sin} m phi) is a tall-skinny,
// block-diagonal contraction over particles k.  Each pass handles P particles:
//   phase 1  thread = particle: all R (n1*(lmax+1) values) and Y (L pairs) features -> shared memory
//            sR[feature][k] (row stride P+2 doubles), sY[pair][k] as (cos,sin) double2 (row stride P+1)
//   phase 2  lane = unit (l, m, n-chunk of NCH): 2*NCH register accumulators (cos and sin columns);
//            a group of WG warps covers all units for its slice of the pass's particles, reading two
//            particles per LDS.128; operands of lanes that share a level are shared-memory broadcasts.
// Accumulators persist over all passes of the block; at the end the G groups are combined in a fixed order
// and the block writes one partial table (2T doubles) to the workspace.
// =========================================================================================================
struct CoeffPlan {
    int nmax, lmax, n1, L, T;
    int nR;          // radial feature rows = n1*(lmax+1)
    int P;           // particles per pass
    int G, WG;       // groups per block, warps per group
    int nchunks;     // n-chunks per (l,m) pair
    int units;       // L*nchunks
    int rstride;     // doubles per sR row
    int ystride;     // double2 per sY row
    int blocks;      // grid size
    long long passes;            // total passes = ceil(N/P)
    long long passes_per_block;  // contiguous passes per block
    size_t smem_bytes;
};

template <int LMAX, int NCH>
__global__ void __launch_bounds__(256)
scf_accumulate_kernel(const double* __restrict__ pos, const double* __restrict__ mass, long long N,
                      CoeffPlan pl, double* __restrict__ partial) {
    extern __shared__ __align__(16) double smem[];
    double* sR = smem;
    double2* sY = reinterpret_cast<double2*>(smem + (size_t)pl.nR * pl.rstride);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n1 = pl.n1;

    // ---- phase-2 role of this lane ---------------------------------------------------------------------
    const int grp = warp / pl.WG, wsub = warp - grp * pl.WG;
    int unit = wsub * 32 + lane;
    const bool active = (unit < pl.units) && (grp < pl.G);
    if (!active) unit = 0;
    const int uj = unit / pl.nchunks, uc = unit - uj * pl.nchunks;
    int ul = 0;
    while (lm_index(ul + 1, 0) <= uj) ++ul;
    const int un0 = uc * NCH;
    const int unn = min(NCH, n1 - un0);
    const double* rrow = sR + (size_t)(ul * n1 + un0) * pl.rstride;
    const double2* yrow = sY + (size_t)uj * pl.ystride;
    const int kper = pl.P / pl.G;
    const int kbeg = (grp < pl.G ? grp : 0) * kper, kend = kbeg + kper;

    double ac[NCH], as[NCH];
#pragma unroll
    for (int i = 0; i < NCH; ++i) { ac[i] = 0.0; as[i] = 0.0; }

    const long long pass0 = (long long)blockIdx.x * pl.passes_per_block;
    const long long pass1 = min(pl.passes, pass0 + pl.passes_per_block);

    for (long long pass = pass0; pass < pass1; ++pass) {
        // ---- phase 1: features of particle k ------------------------------------------------------------
        if (tid < pl.P) {
            const long long k = pass * pl.P + tid;
            double x = 1.0, y = 0.0, z = 0.0, mk = 0.0;   // padding particles carry zero mass
            if (k < N) { x = pos[k]; y = pos[N + k]; z = pos[2 * N + k]; mk = mass[k]; }
            const Geom g = geometry(x, y, z);

            // radial: R_l[n] = m_k f_l C_n^(2l+3/2)(xi)
            const double u = 1.0 / (1.0 + g.r);
            const double xi = (g.r - 1.0) * u;
            const double s = g.r * u * u;
            double fl = -u * mk;
            double* rp = sR + tid;
#pragma unroll 1
            for (int l = 0; l <= LMAX; ++l) {
                double C = 1.0, Cm = 0.0;
                for (int n = 0; n < n1; ++n) {
                    rp[0] = fl * C;
                    rp += pl.rstride;
                    const double a = c_basis.geg_a[l][n + 1], b = c_basis.geg_b[l][n + 1];
                    const double Cn = fma(a * xi, C, -b * Cm);
                    Cm = C; C = Cn;
                }
                fl *= s;
            }

            // angular: Y_lm = P_lm (cos m phi, sin m phi)
            double cm[LMAX + 1], sm[LMAX + 1];
            cm[0] = 1.0; sm[0] = 0.0;
#pragma unroll
            for (int m = 1; m <= LMAX; ++m) {
                cm[m] = fma(cm[m - 1], g.cp, -sm[m - 1] * g.sp);
                sm[m] = fma(sm[m - 1], g.cp, cm[m - 1] * g.sp);
            }
            double U1[LMAX + 1], U2[LMAX + 1];
            double2* yp = sY + tid;
#pragma unroll
            for (int l = 0; l <= LMAX; ++l) {
                double U0[LMAX + 1];
                if (l == 0) {
                    U0[0] = 1.0;
                } else if (l == 1) {
                    U0[0] = g.ct; U0[1] = 1.0;
                } else {
#pragma unroll
                    for (int m = 0; m <= l - 2; ++m) {
                        const double a = double(2 * l - 1) / double(l - m), b = double(l + m - 1) / double(l - m);
                        U0[m] = fma(a * g.ct, U1[m], -b * U2[m]);
                    }
                    U0[l - 1] = double(2 * l - 1) * g.ct * U1[l - 1];
                    U0[l] = double(2 * l - 1) * g.st * U1[l - 1];
                }
#pragma unroll
                for (int m = 0; m <= l; ++m) {
                    const double p = (m == 0) ? U0[0] : g.st * U0[m];
                    yp[(size_t)lm_index(l, m) * pl.ystride] = make_double2(p * cm[m], p * sm[m]);
                }
#pragma unroll
                for (int m = 0; m <= l; ++m) { U2[m] = U1[m]; U1[m] = U0[m]; }
            }
        }
        __syncthreads();

        // ---- phase 2: register-tiled accumulation, two particles per shared-memory load -------------------
        if (active) {
            for (int k = kbeg; k < kend; k += 2) {
                const double2 y0 = yrow[k], y1 = yrow[k + 1];
#pragma unroll
                for (int i = 0; i < NCH; ++i) {
                    const double2 r = *reinterpret_cast<const double2*>(rrow + (size_t)i * pl.rstride + k);
                    ac[i] = fma(r.x, y0.x, ac[i]);
                    as[i] = fma(r.x, y0.y, as[i]);
                    ac[i] = fma(r.y, y1.x, ac[i]);
                    as[i] = fma(r.y, y1.y, as[i]);
                }
            }
        }
        __syncthreads();
    }

    // ---- combine the G groups in a fixed order; one partial table per block -----------------------------
    double* sOut = smem;   // [G][2T]
    if (active) {
#pragma unroll
        for (int i = 0; i < NCH; ++i)
            if (i < unn) {
                sOut[(size_t)grp * 2 * pl.T + (un0 + i) * pl.L + uj] = ac[i];
                sOut[(size_t)grp * 2 * pl.T + pl.T + (un0 + i) * pl.L + uj] = as[i];
            }
    }
    __syncthreads();
    for (int t = tid; t < 2 * pl.T; t += blockDim.x) {
        double v = sOut[t];
        for (int gI = 1; gI < pl.G; ++gI) v += sOut[(size_t)gI * 2 * pl.T + t];
        partial[(size_t)blockIdx.x * 2 * pl.T + t] = v;
    }
}

// S5: fixed-order reduction over block partials and normalisation.
__global__ void __launch_bounds__(128)
scf_finalize_kernel(const double* __restrict__ partial, int blocks, int nmax, int lmax,
                    double* __restrict__ A, double* __restrict__ B) {
    const int L = num_lm(lmax), T = (nmax + 1) * L;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * T) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int b = 0;
    for (; b + 3 < blocks; b += 4) {
        s0 += partial[(size_t)(b + 0) * 2 * T + t];
        s1 += partial[(size_t)(b + 1) * 2 * T + t];
        s2 += partial[(size_t)(b + 2) * 2 * T + t];
        s3 += partial[(size_t)(b + 3) * 2 * T + t];
    }
    for (; b < blocks; ++b) s0 += partial[(size_t)b * 2 * T + t];
    const double sum = (s0 + s1) + (s2 + s3);
    const int tt = (t < T) ? t : t - T;
    const int n = tt / L, j = tt - n * L;
    int l = 0;
    while (lm_index(l + 1, 0) <= j) ++l;
    const int m = j - lm_index(l, 0);
    const double norm = c_basis.norm_nl[l][n] * c_basis.N_lm[j];
    if (t < T) A[tt] = norm * sum;
    else B[tt] = (m == 0) ? 0.0 : norm * sum;
}

// ---------------------------------------------------------------------------------------------------------
// Host side: plan, workspace, launches.
// ---------------------------------------------------------------------------------------------------------
constexpr int kCoeffNCH = 11;
constexpr int kCoeffMaxBlocks = 148 * 4;
constexpr size_t kSmemBudget = 227 * 1024;

static CoeffPlan make_coeff_plan(long long N, int nmax, int lmax) {
    CoeffPlan p{};
    p.nmax = nmax; p.lmax = lmax; p.n1 = nmax + 1; p.L = num_lm(lmax); p.T = p.n1 * p.L;
    p.nR = p.n1 * (lmax + 1);
    p.nchunks = (p.n1 + kCoeffNCH - 1) / kCoeffNCH;
    p.units = p.L * p.nchunks;
    p.WG = (p.units + 31) / 32;
    // Choose P (multiple of 32, <= 128) and G so that G*WG warps >= P/32 where possible and the features fit.
    auto smem_for = [&](int P) {
        // slack rows: lanes of a short last n-chunk read (and ignore) rows past their level
        const int slack = p.nchunks * kCoeffNCH - p.n1;
        size_t r = (size_t)(p.nR + slack) * (P + 2) * 8 + (size_t)p.L * (P + 1) * 16;
        size_t out = (size_t)2 * p.T * 8 * 8;   // room for up to 8 groups in the final combine
        return r > out ? r : out;
    };
    int P = 64;
    while (P > 32 && smem_for(P) > kSmemBudget / 3) P -= 32;          // prefer >= 3 blocks per SM
    if (smem_for(P) > kSmemBudget / 3) { P = 64; while (P > 32 && smem_for(P) > kSmemBudget) P -= 32; }
    p.P = P;
    int G = (P / 32 + p.WG - 1) / p.WG;       // enough warps that every phase-1 thread exists
    if (G < 1) G = 1;
    while ((P / 2) % G != 0) ++G;             // each group gets an even number of particles
    if (G > 8) G = 8;
    p.G = G;
    p.rstride = P + 2;
    p.ystride = P + 1;
    p.smem_bytes = smem_for(P);
    p.passes = (N + P - 1) / P;
    long long blocks = p.passes < kCoeffMaxBlocks ? p.passes : kCoeffMaxBlocks;
    p.passes_per_block = (p.passes + blocks - 1) / blocks;
    p.blocks = (int)((p.passes + p.passes_per_block - 1) / p.passes_per_block);
    return p;
}

size_t scf_coeffs_workspace(long long N, int nmax, int lmax) {
    CoeffPlan p = make_coeff_plan(N, nmax, lmax);
    return round_up((size_t)p.blocks * 2 * p.T * sizeof(double), 256);
}

template <int LMAX>
static cudaError_t launch_accumulate(const double* pos, const double* mass, long long N, const CoeffPlan& p,
                                     double* partial, cudaStream_t st) {
    auto kern = scf_accumulate_kernel<LMAX, kCoeffNCH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_bytes);
    if (e != cudaSuccess) return e;
    int threads = 32 * p.G * p.WG;
    if (threads < p.P) threads = p.P;
    kern<<<p.blocks, threads, p.smem_bytes, st>>>(pos, mass, N, p, partial);
    return cudaGetLastError();
}

cudaError_t scf_coeffs_launch(const double* pos, const double* mass, long long N, int nmax, int lmax,
                              double* A, double* B, void* ws, cudaStream_t st) {
    cudaError_t e = etics_upload_constants();
    if (e != cudaSuccess) return e;
    const CoeffPlan p = make_coeff_plan(N, nmax, lmax);
    double* partial = static_cast<double*>(ws);
    switch (lmax) {
#define ETICS_CASE(LM) case LM: e = launch_accumulate<LM>(pos, mass, N, p, partial, st); break;
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5)
        ETICS_CASE(6) ETICS_CASE(7) ETICS_CASE(8) ETICS_CASE(9) ETICS_CASE(10)
#undef ETICS_CASE
        default: return cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) return e;
    const int T2 = 2 * p.T;
    scf_finalize_kernel<<<(T2 + 127) / 128, 128, 0, st>>>(partial, p.blocks, nmax, lmax, A, B);
    return cudaGetLastError();
}

template <int LMAX>
static cudaError_t launch_eval(const double* pos, long long N, int nmax, const double* A, const double* B,
                               double* acc, double* pot, cudaStream_t st) {
    auto kern = scf_eval_kernel<LMAX>;
    const size_t smem = (size_t)(nmax + 1) * num_lm(LMAX) * sizeof(double2);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long blocks = (N + kEvalThreads - 1) / kEvalThreads;
    kern<<<(unsigned)blocks, kEvalThreads, smem, st>>>(pos, N, nmax, A, B, acc, pot);
    return cudaGetLastError();
}

cudaError_t scf_force_launch(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                             double* acc, double* pot, cudaStream_t st) {
    cudaError_t e = etics_upload_constants();
    if (e != cudaSuccess) return e;
    switch (lmax) {
#define ETICS_CASE(LM) case LM: return launch_eval<LM>(pos, N, nmax, A, B, acc, pot, st);
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5)
        ETICS_CASE(6) ETICS_CASE(7) ETICS_CASE(8) ETICS_CASE(9) ETICS_CASE(10)
#undef ETICS_CASE
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace etics

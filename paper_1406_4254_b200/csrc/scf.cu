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
// Per level l the sums S_l[n][f] = sum_k R_l[k][n] Y_l[k][f] form a tall-skinny contraction over particles k:
//   R_l[k][n] = m_k Phi~_nl(r_k)                                   (n1 = nmax+1 radial features per level)
//   Y_l[k][f] = P_l0 | P_lm cos m phi | P_lm sin m phi              (2l+1 real angular features per level,
//               f = 0 -> (m=0), f = 2m-1 -> cos, f = 2m -> sin)
// Not tensor-core work (north_star); the fp64 FMA pipe is the roof, so the job is to feed it from registers.
// Each pass handles P particles:
//   phase 1  thread = particle: geometry, Gegenbauer and Legendre/trig recurrences in registers; features to
//            shared memory, one row per feature, particles contiguous (sR[row][k], sY[row][k], row stride P+2).
//   phase 2  thread = unit (n-chunk of NCH, level l, tile of YT consecutive angular features): a register
//            tile of NCH x YT accumulators; per two particles NCH + YT LDS.128 feed 2*NCH*YT FMAs.  The block's
//            threads form `streams` copies of the unit list, each taking its own slice of the pass.
// Accumulators persist over all passes of the block; at the end the streams are combined in ascending order
// and the block writes one partial table (2T doubles) to the workspace (no atomics: deterministic).
// =========================================================================================================
// gamma_lm of the monic Legendre recurrence q_l = ct q_{l-1} - gamma_lm q_{l-2} (column m, l >= m+2)
__host__ __device__ constexpr double leg_gamma_c(int l, int m) {
    return (l >= m + 2) ? double((l + m - 1) * (l - 1 - m)) / double((2 * l - 1) * (2 * l - 3)) : 0.0;
}

// Angular rows of column M for one particle: q_M = st^M, q_l = ct q_{l-1} - gamma q_{l-2};
// rows of level l: q_l0 at l^2, (q_lM cos M phi, q_lM sin M phi) at l^2 + 2M - 1, l^2 + 2M.  yk = sY + k.
template <int LMAX, int M>
__device__ __forceinline__ void scf_angular_column(double ct, double st, double cp, double sp, double* yk, int stride) {
    double cm = 1.0, sm = 0.0, q1 = 1.0, q2 = 0.0;
#pragma unroll
    for (int i = 1; i <= M; ++i) {
        const double c2 = fma(cm, cp, -sm * sp);
        sm = fma(sm, cp, cm * sp);
        cm = c2;
        q1 *= st;
    }
#pragma unroll
    for (int l = M; l <= LMAX; ++l) {
        if (M == 0) {
            yk[(l * l) * stride] = q1;
        } else {
            yk[(l * l + 2 * M - 1) * stride] = q1 * cm;
            yk[(l * l + 2 * M) * stride] = q1 * sm;
        }
        if (l < LMAX) {
            const double qn = (l == M) ? ct * q1 : fma(ct, q1, -leg_gamma_c(l + 1, M) * q2);
            q2 = q1; q1 = qn;
        }
    }
}

template <int LMAX, int M>
__device__ __forceinline__ void scf_angular_dispatch(int row0, int rmask, double ct, double st, double cp, double sp,
                                                     double* yk, int stride) {
    if constexpr (M <= LMAX) {
        if ((M & rmask) == row0) scf_angular_column<LMAX, M>(ct, st, cp, sp, yk, stride);
        scf_angular_dispatch<LMAX, M + 1>(row0, rmask, ct, st, cp, sp, yk, stride);
    }
}

// Radial rows of level LV for one particle: monic Gegenbauer Q_n scaled by m_k f_l:
// R_0 = m f_l, R_1 = xi R_0, R_n = xi R_{n-1} - beta_n R_{n-2}.  rk = sR + k.
template <int LV>
__device__ __forceinline__ void scf_radial_level(double f0, double xi, double sv, int n1, const double* __restrict__ beta,
                                                 double* rk, int stride) {
    double r0 = f0;
#pragma unroll
    for (int i = 0; i < LV; ++i) r0 *= sv;
    double* rp = rk + (LV * n1) * stride;
    double r1 = xi * r0;
    rp[0] = r0;
    if (n1 > 1) rp[stride] = r1;
    int n = 2;
#pragma unroll 2
    for (; n + 1 < n1; n += 2) {
        r0 = fma(xi, r1, -beta[n] * r0);
        rp[n * stride] = r0;
        r1 = fma(xi, r0, -beta[n + 1] * r1);
        rp[(n + 1) * stride] = r1;
    }
    if (n < n1) rp[n * stride] = fma(xi, r1, -beta[n] * r0);
}

template <int LMAX, int LV>
__device__ __forceinline__ void scf_radial_dispatch(int row0, int rmask, double f0, double xi, double sv, int n1,
                                                    double* rk, int stride) {
    if constexpr (LV <= LMAX) {
        if ((LV & rmask) == row0) scf_radial_level<LV>(f0, xi, sv, n1, c_basis.geg_beta[LV], rk, stride);
        scf_radial_dispatch<LMAX, LV + 1>(row0, rmask, f0, xi, sv, n1, rk, stride);
    }
}

constexpr int kCoeffThreads = 256;
constexpr int kCoeffNCH = 11;   // radial features per unit
constexpr int kCoeffYT = 4;     // angular features per unit

struct CoeffPlan {
    int nmax, lmax, n1, L, T;
    int nR, nY;      // feature rows: n1*(lmax+1) radial (+slack), (lmax+1)^2 angular (+slack)
    int P;           // particles per pass
    int UL;          // units per n-chunk = sum_l ceil((2l+1)/YT)
    int nchunks, units, streams;
    int kper;        // particles per stream per pass (even)
    int stride;      // doubles per feature row
    int max_blocks;  // workspace is sized for this many block partials
    long long passes;
    size_t smem_bytes;
};

template <int LMAX>
__global__ void __launch_bounds__(kCoeffThreads, 2)
scf_accumulate_kernel(const double* __restrict__ pos, const double* __restrict__ mass, long long N,
                      CoeffPlan pl, long long passes_per_block, double* __restrict__ partial) {
    constexpr int NCH = kCoeffNCH, YT = kCoeffYT;
    extern __shared__ __align__(16) double smem[];
    double* sR = smem;
    double* sY = smem + (size_t)pl.nR * pl.stride;

    const int tid = threadIdx.x;
    const int n1 = pl.n1, stride = pl.stride;

    // ---- phase-2 role of this thread -------------------------------------------------------------------
    const int strm = tid / pl.units;
    const bool active = strm < pl.streams;
    const int unit = active ? tid - strm * pl.units : 0;
    const int uc = unit / pl.UL;                  // n-chunk
    int uv = unit - uc * pl.UL, ul = 0;           // level and feature tile
    while (uv >= (2 * ul + 1 + YT - 1) / YT) { uv -= (2 * ul + 1 + YT - 1) / YT; ++ul; }
    const int un0 = uc * NCH, uf0 = uv * YT;
    // the stream's slice of the pass: pairs [s*(P/2)/streams, (s+1)*(P/2)/streams)
    const int kbeg = 2 * (((active ? strm : 0) * (pl.P / 2)) / pl.streams);
    const int kcnt = 2 * ((((active ? strm : 0) + 1) * (pl.P / 2)) / pl.streams) - kbeg;
    const double* rrow = sR + (size_t)(ul * n1 + un0) * stride + kbeg;
    const double* yrow = sY + (size_t)(ul * ul + uf0) * stride + kbeg;

    double acc[NCH][YT];
#pragma unroll
    for (int i = 0; i < NCH; ++i)
#pragma unroll
        for (int j = 0; j < YT; ++j) acc[i][j] = 0.0;

    const long long pass0 = (long long)blockIdx.x * passes_per_block;
    const long long pass1 = min(pl.passes, pass0 + passes_per_block);

    double* sG = sY + (size_t)pl.nY * stride;   // geometry, double-buffered: 2 x 8 fields x P
    const int P = pl.P;                          // 32, 64 or 128: tasks (row, k) need no division
    const int task_k = tid & (P - 1);
    const int task_row0 = tid / P, task_rmask = kCoeffThreads / P - 1;   // rows row0, row0 + 256/P, ...

    // geometry of particle k of a pass (thread = particle), into buffer `buf`
    auto phase0 = [&](long long pass, int buf) {
        if (tid < P && pass < pass1) {
            double* G = sG + buf * 8 * P;
            const long long k = pass * P + tid;
            double x = 1.0, y = 0.0, z = 0.0, mk = 0.0;   // padding particles carry zero mass
            if (k < N) { x = pos[k]; y = pos[N + k]; z = pos[2 * N + k]; mk = mass[k]; }
            const Geom g = geometry(x, y, z);
            const double u = 1.0 / (1.0 + g.r);
            G[0 * P + tid] = -u * mk;              // m_k f_0,  f_l = -u s^l
            G[1 * P + tid] = (g.r - 1.0) * u;      // xi
            G[2 * P + tid] = g.r * u * u;          // s
            G[3 * P + tid] = g.ct;
            G[4 * P + tid] = g.st;
            G[5 * P + tid] = g.cp;
            G[6 * P + tid] = g.sp;
        }
    };
    phase0(pass0, 0);
    __syncthreads();

    for (long long pass = pass0; pass < pass1; ++pass) {
        const int buf = (int)((pass - pass0) & 1);
        // ---- phase 1: feature rows of this pass; task = (row, particle k), the row is warp-uniform ------------
        {
            const double* G = sG + buf * 8 * P;
            scf_radial_dispatch<LMAX, 0>(task_row0, task_rmask, G[0 * P + task_k], G[1 * P + task_k], G[2 * P + task_k],
                                         n1, sR + task_k, stride);
            scf_angular_dispatch<LMAX, 0>(task_row0, task_rmask, G[3 * P + task_k], G[4 * P + task_k], G[5 * P + task_k],
                                          G[6 * P + task_k], sY + task_k, stride);
        }
        __syncthreads();
        // ---- phase 0 of the next pass (overlaps phase 2 of the other warps) ---------------------------------
        phase0(pass + 1, buf ^ 1);

        // ---- phase 2: register-tiled accumulation, two particles per shared-memory load -------------------
        if (active) {
#pragma unroll 1
            for (int k = 0; k < kcnt; k += 2) {
                double2 yv[YT];
#pragma unroll
                for (int j = 0; j < YT; ++j) yv[j] = *reinterpret_cast<const double2*>(yrow + (size_t)j * stride + k);
#pragma unroll
                for (int i = 0; i < NCH; ++i) {
                    const double2 r = *reinterpret_cast<const double2*>(rrow + (size_t)i * stride + k);
#pragma unroll
                    for (int j = 0; j < YT; ++j) {
                        acc[i][j] = fma(r.x, yv[j].x, acc[i][j]);
                        acc[i][j] = fma(r.y, yv[j].y, acc[i][j]);
                    }
                }
            }
        }
        __syncthreads();
    }

    // ---- combine the streams in ascending order; one partial table per block ----------------------------
    double* sOut = smem;   // [2T]: cos table then sin table
    for (int t = tid; t < 2 * pl.T; t += kCoeffThreads) sOut[t] = 0.0;
    __syncthreads();
    for (int sI = 0; sI < pl.streams; ++sI) {
        if (active && strm == sI) {
#pragma unroll
            for (int i = 0; i < NCH; ++i)
#pragma unroll
                for (int j = 0; j < YT; ++j) {
                    const int n = un0 + i, f = uf0 + j;
                    if (n < n1 && f <= 2 * ul) {
                        const int m = (f + 1) >> 1;
                        const bool is_sin = (f > 0) && ((f & 1) == 0);
                        sOut[(is_sin ? pl.T : 0) + n * pl.L + lm_index(ul, m)] += acc[i][j];
                    }
                }
        }
        __syncthreads();
    }
    for (int t = tid; t < 2 * pl.T; t += kCoeffThreads) partial[(size_t)blockIdx.x * 2 * pl.T + t] = sOut[t];
}

// S5: fixed-order reduction over block partials and normalisation.
// Block = 32 outputs (threadIdx.x, coalesced along the table) x kFinSlices slices of the block partials
// (threadIdx.y); every slice sums its partials b = y, y + kFinSlices, ... in ascending order with four
// interleaved accumulators, then the slices are combined in ascending y.  The order depends only on `blocks`.
constexpr int kFinSlices = 16;

__global__ void __launch_bounds__(32 * kFinSlices)
scf_finalize_kernel(const double* __restrict__ partial, int blocks, int nmax, int lmax,
                    double* __restrict__ A, double* __restrict__ B) {
    __shared__ double sh[kFinSlices][33];
    const int L = num_lm(lmax), T = (nmax + 1) * L;
    const int t = blockIdx.x * 32 + threadIdx.x, y = threadIdx.y;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    if (t < 2 * T) {
        int b = y;
        for (; b + 3 * kFinSlices < blocks; b += 4 * kFinSlices) {
            s0 += partial[(size_t)(b + 0 * kFinSlices) * 2 * T + t];
            s1 += partial[(size_t)(b + 1 * kFinSlices) * 2 * T + t];
            s2 += partial[(size_t)(b + 2 * kFinSlices) * 2 * T + t];
            s3 += partial[(size_t)(b + 3 * kFinSlices) * 2 * T + t];
        }
        for (; b < blocks; b += kFinSlices) s0 += partial[(size_t)b * 2 * T + t];
    }
    sh[y][threadIdx.x] = (s0 + s1) + (s2 + s3);
    __syncthreads();
    if (y != 0 || t >= 2 * T) return;
    double sum = 0.0;
#pragma unroll
    for (int i = 0; i < kFinSlices; ++i) sum += sh[i][threadIdx.x];
    const int tt = (t < T) ? t : t - T;
    const int n = tt / L, j = tt - n * L;
    int l = 0;
    while (lm_index(l + 1, 0) <= j) ++l;
    const int m = j - lm_index(l, 0);
    const double norm = (c_basis.norm_nl[l][n] * c_basis.geg_scale[l][n]) * (c_basis.N_lm[j] * c_basis.leg_scale[l][m]);
    if (t < T) A[tt] = norm * sum;
    else B[tt] = (m == 0) ? 0.0 : norm * sum;
}

// ---------------------------------------------------------------------------------------------------------
// Host side: plan, workspace, launches.
// ---------------------------------------------------------------------------------------------------------
constexpr int kCoeffMaxBlocks = 148 * 8;
constexpr size_t kSmemBudget = 227 * 1024;

static CoeffPlan make_coeff_plan(long long N, int nmax, int lmax) {
    CoeffPlan p{};
    p.nmax = nmax; p.lmax = lmax; p.n1 = nmax + 1; p.L = num_lm(lmax); p.T = p.n1 * p.L;
    p.nchunks = (p.n1 + kCoeffNCH - 1) / kCoeffNCH;
    p.UL = 0;
    for (int l = 0; l <= lmax; ++l) p.UL += (2 * l + 1 + kCoeffYT - 1) / kCoeffYT;
    p.units = p.UL * p.nchunks;
    // slack rows: the last n-chunk / feature tile of a level reads (and ignores) rows past its level
    p.nR = p.n1 * (lmax + 1) + (p.nchunks * kCoeffNCH - p.n1);
    p.nY = (lmax + 1) * (lmax + 1) + (kCoeffYT - 1);
    auto smem_for = [&](int P) { return ((size_t)(p.nR + p.nY) * (P + 2) + (size_t)16 * P) * sizeof(double); };
    // P in {128, 64, 32}: the largest that leaves two resident blocks per SM (registers allow two), else the
    // largest that fits at all
    int P = 128;
    while (P > 32 && smem_for(P) > kSmemBudget / 2) P /= 2;
    if (smem_for(P) > kSmemBudget / 2) { P = 128; while (P > 32 && smem_for(P) > kSmemBudget) P /= 2; }
    int streams = kCoeffThreads / p.units;
    if (streams < 1) streams = 1;
    if (streams > P / 2) streams = P / 2;
    p.P = P; p.streams = streams; p.kper = 0;
    p.stride = P + 2;
    p.smem_bytes = smem_for(P);
    p.passes = (N + P - 1) / P;
    p.max_blocks = (int)(p.passes < kCoeffMaxBlocks ? p.passes : kCoeffMaxBlocks);
    return p;
}

size_t scf_coeffs_workspace(long long N, int nmax, int lmax) {
    CoeffPlan p = make_coeff_plan(N, nmax, lmax);
    return round_up((size_t)p.max_blocks * 2 * p.T * sizeof(double), 256);
}

template <int LMAX>
static cudaError_t launch_accumulate(const double* pos, const double* mass, long long N, const CoeffPlan& p,
                                     double* partial, int* blocks_out, cudaStream_t st) {
    auto kern = scf_accumulate_kernel<LMAX>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_bytes);
    if (e != cudaSuccess) return e;
    // one wave of resident blocks: grid = SMs x blocks per SM (capped by the workspace and by the work)
    int dev = 0, sms = 0, occ = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kCoeffThreads, p.smem_bytes)) != cudaSuccess) return e;
    long long blocks = (long long)sms * (occ > 0 ? occ : 1);
    if (blocks > p.max_blocks) blocks = p.max_blocks;
    const long long ppb = (p.passes + blocks - 1) / blocks;
    blocks = (p.passes + ppb - 1) / ppb;
    *blocks_out = (int)blocks;
    kern<<<(unsigned)blocks, kCoeffThreads, p.smem_bytes, st>>>(pos, mass, N, p, ppb, partial);
    return cudaGetLastError();
}

cudaError_t scf_coeffs_launch(const double* pos, const double* mass, long long N, int nmax, int lmax,
                              double* A, double* B, void* ws, cudaStream_t st) {
    cudaError_t e = etics_upload_constants();
    if (e != cudaSuccess) return e;
    const CoeffPlan p = make_coeff_plan(N, nmax, lmax);
    double* partial = static_cast<double*>(ws);
    int blocks = 0;
    switch (lmax) {
#define ETICS_CASE(LM) case LM: e = launch_accumulate<LM>(pos, mass, N, p, partial, &blocks, st); break;
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5)
        ETICS_CASE(6) ETICS_CASE(7) ETICS_CASE(8) ETICS_CASE(9) ETICS_CASE(10)
#undef ETICS_CASE
        default: return cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) return e;
    const int T2 = 2 * p.T;
    scf_finalize_kernel<<<(T2 + 31) / 32, dim3(32, kFinSlices), 0, st>>>(partial, blocks, nmax, lmax, A, B);
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

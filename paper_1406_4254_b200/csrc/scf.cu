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

cudaError_t scf_init_constants();

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
// threads per block: 64: 166 us, 128: 148.5, 256: 145.4, 512: 162.6 at (10,6), N = 1e6; (20,10) at N = 1e7: 128: 6.08 ms, 256: 6.45 ms
__host__ __device__ constexpr int eval_threads(int lmax) { return lmax <= 6 ? 256 : 128; }
__host__ __device__ constexpr bool eval_persistent(int lmax) { return lmax > 6; }
constexpr int kEvalGridPerSM = 8;
#ifndef ETICS_EVAL_MINBLOCKS
#define ETICS_EVAL_MINBLOCKS 2
#endif

// gamma_lm of the monic Legendre recurrence q_l = ct q_{l-1} - gamma_lm q_{l-2} (column m, l >= m+2)
__host__ __device__ constexpr double leg_gamma_c(int l, int m) {
    return (l >= m + 2) ? double((l + m - 1) * (l - 1 - m)) / double((2 * l - 1) * (2 * l - 3)) : 0.0;
}

// Scale of table entry (l, n, m): [0] h_lm = leg_scale[l][m], [1] g_n h_lm = geg_scale[l][n] * leg_scale[l][m] (monic Gegenbauer
// variant).  Written once per device by scf_init_constants, read-only afterwards.
static __device__ double d_pack_scale[2][kMaxL + 1][kMaxN + 1][kMaxL + 1];

// N1C > 0: nmax + 1 known at compile time (the n loops unroll fully and the compiler schedules across them);
// N1C = 0: run-time nmax.
// PO: potential only ("faster since the derivatives ... are not calculated") — no C'_n chain, no
// dP/dtheta, no U_lm sums, no transform; acc is not touched.  Otherwise both are computed; pot == nullptr (force only)
// skips the store of the potential.
template <int LMAX, int N1C, bool PO>
__global__ void __launch_bounds__(eval_threads(LMAX), LMAX <= 6 ? ETICS_EVAL_MINBLOCKS : 1)
scf_eval_kernel(const double* __restrict__ pos, long long N, int nmax,
                const double* __restrict__ A, const double* __restrict__ B,
                double* __restrict__ acc, double* __restrict__ pot) {
    // Monic Gegenbauer recurrence (scale g_n folded into the table, one multiply less per order) only where the n loops
    // are unrolled — beta_n are then immediate constant-bank operands: 155.5 -> 148.9 us at (10,6), N = 1e6; with a
    // run-time loop the same change was slower (164 -> 171 us).
    constexpr bool kMonicGeg = N1C > 0;
    extern __shared__ double2 s_tab[];   // (A,B) pairs, index n1*l(l+1)/2 + n*(l+1) + m
    constexpr int L = num_lm(LMAX);
    const int n1 = N1C > 0 ? N1C : nmax + 1;
    constexpr int kEvalThreads = eval_threads(LMAX);
    // one-shot blocks: the particle's position is asked for before the table repack, so that the DRAM round trip runs under it
    const long long k1 = (long long)blockIdx.x * kEvalThreads + threadIdx.x;
    double x1 = 1.0, y1 = 0.0, z1 = 0.0;
    if (!eval_persistent(LMAX) && k1 < N) { x1 = pos[k1]; y1 = pos[N + k1]; z1 = pos[2 * N + k1]; }
    for (int g = threadIdx.x; g < n1 * L; g += kEvalThreads) {
        const int n = g / L, j = g - n * L;
        int l = 0;
        while (lm_index(l + 1, 0) <= j) ++l;
        const int m = j - lm_index(l, 0);
        // monic recurrences below: C_n = g_n Q_n, P_lm = h_lm q_lm; the scales ride on the coefficients
        // (from a table in GLOBAL memory: the lanes ask for different (l, n, m), and a constant-bank load with 32 different
        // addresses is replayed 32 times — with c_basis here the repack was 17 % of the kernel's stall samples at N = 1e6)
        const double sc = d_pack_scale[kMonicGeg ? 1 : 0][l][n][m];
        s_tab[n1 * lm_index(l, 0) + n * (l + 1) + m] = make_double2(A[g] * sc, B[g] * sc);
    }
    __syncthreads();

    auto evaluate = [&](const long long k, const double px, const double py, const double pz) {
    const Geom g = geometry(px, py, pz);

    // cos(m phi), sin(m phi): parked in lane-private shared-memory columns while the n loops run, so that the
    // 4 (l+1) running sums of a level and the two previous angular rows have the registers to themselves
    double* s_trig = reinterpret_cast<double*>(s_tab + n1 * L) + threadIdx.x;
    {
        double c = 1.0, sn = 0.0;
#pragma unroll
        for (int m = 1; m <= LMAX; ++m) {
            const double c2 = fma(c, g.cp, -sn * g.sp);
            sn = fma(sn, g.cp, c * g.sp);
            c = c2;
            s_trig[(2 * m) * kEvalThreads] = c;
            s_trig[(2 * m + 1) * kEvalThreads] = sn;
        }
    }

    const double u = __drcp_rn(1.0 + g.r);
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
            for (int m = 0; m <= l - 2; ++m) U0[m] = fma(g.ct, U1[m], -leg_gamma_c(l, m) * U2[m]);
            U0[l - 1] = g.ct * U1[l - 1];
            U0[l] = g.st * U1[l - 1];
        }
        // ---- radial sums over n -----------------------------------------------------------------------
        double sa[LMAX + 1], sad[LMAX + 1], sb[LMAX + 1], sbd[LMAX + 1];
#pragma unroll
        for (int m = 0; m <= l; ++m) { sa[m] = 0.0; sad[m] = 0.0; sb[m] = 0.0; sbd[m] = 0.0; }
        double C = 1.0, Cm = 0.0, D = 0.0, Dm = 0.0;   // monic Q_n, Q_{n-1}, dQ_n/dxi, dQ_{n-1}/dxi
        const double* __restrict__ beta = c_basis.geg_beta[l];
#pragma unroll(N1C == 0 ? 4 : N1C > 16 ? 3 : 32)
        for (int n = 0; n < (N1C > 0 ? N1C : n1); ++n) {
#pragma unroll
            for (int m = 0; m <= l; ++m) {
                const double2 ab = tl[n * (l + 1) + m];
                sa[m] = fma(ab.x, C, sa[m]);
                if (!PO) sad[m] = fma(ab.x, D, sad[m]);
                if (m > 0) {
                    sb[m] = fma(ab.y, C, sb[m]);
                    if (!PO) sbd[m] = fma(ab.y, D, sbd[m]);
                }
            }
            // Q_{n+1} = xi Q_n - beta_{n+1} Q_{n-1};  Q'_{n+1} = xi Q'_n + Q_n - beta_{n+1} Q'_{n-1}
            double Cn, Dn;
            if (kMonicGeg) {
                const double nb = -beta[n + 1];
                Cn = fma(xi, C, nb * Cm);
                Dn = PO ? 0.0 : fma(xi, D, fma(nb, Dm, C));
            } else {
                const double a = c_basis.geg_a[l][n + 1], b = c_basis.geg_b[l][n + 1];
                const double ax = a * xi;
                Cn = fma(ax, C, -b * Cm);
                Dn = PO ? 0.0 : fma(ax, D, fma(a, C, -b * Dm));
            }
            Cm = C; C = Cn; Dm = D; D = Dn;
        }
        tl += n1 * (l + 1);

        // ---- combine the level (P_lm = st U_lm; dP_lm/dtheta = l ct U_lm - (l+m) U_{l-1,m}, dP_l0/dtheta = -st U_l1:
        //      same-column forms, no cancellation near the poles) -------------------------------------------------
        double lv_p = 0.0, lv_r = 0.0, lv_t = 0.0, lv_f = 0.0;
        const double lct = double(l) * g.ct;
#pragma unroll
        for (int m = 0; m <= l; ++m) {
            const double cmm = (m == 0) ? 1.0 : s_trig[(2 * m) * kEvalThreads];
            const double smm = (m == 0) ? 0.0 : s_trig[(2 * m + 1) * kEvalThreads];
            const double Ea = (m == 0) ? sa[0] : fma(sa[m], cmm, sb[m] * smm);
            const double P = (m == 0) ? U0[0] : g.st * U0[m];
            lv_p = fma(P, Ea, lv_p);
            if (PO) continue;
            const double Ed = (m == 0) ? sad[0] : fma(sad[m], cmm, sbd[m] * smm);
            double dP;
            if (m == 0) {
                dP = (l >= 1) ? -(double(l) * g.st) * U0[1] : 0.0;   // -P_l1 / h_l0, h_l1 / h_l0 = l
            } else {
                // in monic terms U_{l-1,m} / h_lm = q_{l-1,m} (l-m)/(2l-1)
                dP = (m < l) ? fma(lct, U0[m], -(double((l + m) * (l - m)) / double(2 * l - 1)) * U1[m]) : lct * U0[m];
            }
            lv_r = fma(P, Ed, lv_r);
            lv_t = fma(dP, Ea, lv_t);
            if (m > 0) {
                const double Fa = fma(sb[m], cmm, -sa[m] * smm);
                lv_f = fma(double(m) * U0[m], Fa, lv_f);
            }
        }
        s_pot = fma(fl, lv_p, s_pot);
        if (!PO) {
            s_r = fma(fl, fma(gl, lv_p, two_u2 * lv_r), s_r);
            s_t = fma(fl, lv_t, s_t);
            s_f = fma(fl, lv_f, s_f);
        }
        fl *= s;
        gl -= xr;
#pragma unroll
        for (int m = 0; m <= l; ++m) { U2[m] = U1[m]; U1[m] = U0[m]; }
    }

    if (!PO) {
        double ax, ay, az;
        to_cartesian(g, -s_r, -s_t * g.rinv, -s_f * g.rinv, ax, ay, az);
        acc[k] = ax;
        acc[N + k] = ay;
        acc[2 * N + k] = az;
    }
    if (PO || pot != nullptr) pot[k] = s_pot;
    };
    if constexpr (eval_persistent(LMAX)) {
        // the grid is a few blocks per SM: a block repacks the table once and then takes particles k, k + gridDim.x * threads, ...
        // ((20,10), N = 1e7: 6.08 -> 5.66 ms; at lmax <= 6 the loop costs registers: 138 -> 147 us, so those stay one-shot)
#pragma unroll 1
        for (long long k = (long long)blockIdx.x * kEvalThreads + threadIdx.x; k < N; k += (long long)gridDim.x * kEvalThreads)
            evaluate(k, pos[k], pos[N + k], pos[2 * N + k]);
    } else {
        if (k1 < N) evaluate(k1, x1, y1, z1);
    }
}

// =========================================================================================================
// Coefficient accumulation (S1–S4).
//
// Per level l the sums S_l[n][f] = sum_k R_l[k][n] Y_l[k][f] form a tall-skinny contraction over particles k:
//   R_l[k][n] = m_k Phi~_nl(r_k)                                   (n1 = nmax+1 radial features per level)
//   Y_l[k][f] = P_l0 | P_lm cos m phi | P_lm sin m phi              (2l+1 real angular features per level,
//               f = 0 -> (m=0), f = 2m-1 -> cos, f = 2m -> sin)
// Not tensor-core work (north_star); the fp64 FMA pipe is the roof, and the shared-memory pipe (128 B/clk/SM =
// 16 doubles per 64 FMAs) is the trap: a feature value that travels through shared memory must feed >= 4 FMAs.
//
// Mapping: WARP = output tile ("unit": level l, W <= 4 consecutive angular features, a chunk of 11 radial
// orders), LANE = particle.  Everything but the particle is warp-uniform, so recurrence coefficients are
// uniform constant-bank operands and every shared-memory access is a fully coalesced, conflict-free row read.
//   phase 0  (warps 0-3, thread = particle, pass p+2): geometry, cos/sin(m phi) -> G (double-buffered)
//   phase 1  (all warps, thread = (particle, column class), pass p+1): monic Legendre columns
//            q_l = ct q_{l-1} - gamma_lm q_{l-2} times cos/sin(m phi) -> Y rows; radial seeds m_k f_l and xi -> F
//   phase 2  (warp = unit, lane = particle, pass p): monic Gegenbauer chain R_n = xi R_{n-1} - beta_n R_{n-2}
//            IN REGISTERS (recomputed by every unit of the level: 2 ops per n against 11 W FMAs — cheaper than
//            sending 11 more rows through shared memory), acc[n][j] += R_n Y_j.
// One barrier per pass; the three phases of an iteration work on different passes, so warps drift apart and the
// latency-bound phases 0/1 overlap the FMA-bound phase 2.  Accumulators persist over all passes of the block;
// at the end the 32 lanes are combined by a fixed butterfly, replicas (small tables) in ascending order, and
// the block writes one partial table (no atomics: deterministic).  Tables with more than 16 units are split into
// unit groups (gridDim.y); a group's blocks recompute phases 0/1 for the levels they need.
// =========================================================================================================
constexpr int kAccThreads = 512;
constexpr int kAccWarps = kAccThreads / 32;
constexpr int kAccP = 128;              // particles per pass
constexpr int kAccSteps = kAccP / 32;   // phase-2 steps per pass (one particle per lane per step)
constexpr int kAccNCH = 11;             // radial orders per unit
constexpr int kAccWMax = 4;             // angular features per unit
constexpr int kAccMaxGroups = 8;
constexpr int kAccGRows = 5 + 2 * kMaxL;   // m f_0, xi, s, ct, st, cos(m phi) m=1..lmax, sin(m phi) m=1..lmax

struct AccUnit { short l, f0, w, n0; };
struct AccGroup {
    int nunits, rep;           // units of this group; replicas per unit (rep * nunits <= 16 warps)
    int la, lb;                // levels whose rows the group needs
    int nrows;                 // feature rows per buffer: Y rows of levels la..lb (row of (l,f) = l^2 + f - la^2),
                               // then one seed row per level, then xi
    AccUnit unit[kAccWarps];
};
struct AccPlan {
    int nmax, lmax, n1, L, T;
    int ngroups;
    int block0;                // first block of this launch (the host entry launches ranges of blocks as their particles arrive)
    long long passes, passes_per_block;
    AccGroup group[kAccMaxGroups];
};

__device__ __forceinline__ double ldc_volatile(const double* p) {
    double v;
    asm volatile("ld.const.f64 %0, [%1];" : "=d"(v) : "l"(__cvta_generic_to_constant(p)));
    return v;
}

// LV >= 0: level known at compile time and n0 == 0, so that every beta_n is a constant-bank operand with an
// immediate offset (no registers held for the recurrence coefficients).  LV < 0: generic (later n-chunks).
template <int W, int LV>
__device__ __forceinline__ void acc_unit_steps(const double* __restrict__ F, const AccGroup& g, const AccUnit u,
                                               int rep, int replica, int lane, double (&acc)[kAccNCH][kAccWMax]) {
    const int l = (LV >= 0) ? LV : u.l;
    const int n0 = (LV >= 0) ? 0 : u.n0;
    const double* __restrict__ beta = c_basis.geg_beta[l];
    const int ny = (g.lb + 1) * (g.lb + 1) - g.la * g.la;   // Y rows of the group
    const double* yb = F + (size_t)(l * l - g.la * g.la + u.f0) * kAccP + lane;
    const double* sb = F + (size_t)(ny + l - g.la) * kAccP + lane;
    const double* xb = F + (size_t)(ny + g.lb - g.la + 1) * kAccP + lane;
    for (int step = replica; step < kAccSteps; step += rep) {
        const int o = step * 32;
        const double xi = xb[o];
        double y[W];
#pragma unroll
        for (int j = 0; j < W; ++j) y[j] = yb[j * kAccP + o];
        double r1 = sb[o], r2 = 0.0;   // R_n, R_{n-1} (R_0 = seed; beta_1 = 0 so that R_1 = xi R_0)
        if (LV < 0) {
            for (int n = 1; n <= n0; ++n) {   // later chunks: run the chain up to their first order
                const double rn = fma(xi, r1, -beta[n] * r2);
                r2 = r1; r1 = rn;
            }
        }
#pragma unroll
        for (int i = 0; i < kAccNCH; ++i) {
#pragma unroll
            for (int j = 0; j < W; ++j) acc[i][j] = fma(r1, y[j], acc[i][j]);
            if (i + 1 < kAccNCH) {
                // the coefficient is re-read from the constant bank at every use (a volatile load cannot be
                // hoisted), so that no register is held for it across the unit's 44 accumulators
                const double rn = (LV >= 0 && i == 0) ? xi * r1 : fma(xi, r1, -ldc_volatile(beta + n0 + i + 1) * r2);
                r2 = r1; r1 = rn;
            }
        }
    }
}

template <int W, int LV = 0>
__device__ __forceinline__ void acc_unit_level(const double* __restrict__ F, const AccGroup& g, const AccUnit u,
                                               int rep, int replica, int lane, double (&acc)[kAccNCH][kAccWMax]) {
    if constexpr (LV > kMaxL) {
        acc_unit_steps<W, -1>(F, g, u, rep, replica, lane, acc);
    } else {
        if (u.n0 == 0 && u.l == LV) {
            if constexpr (W <= 2 * LV + 1) acc_unit_steps<W, LV>(F, g, u, rep, replica, lane, acc);
        } else {
            acc_unit_level<W, LV + 1>(F, g, u, rep, replica, lane, acc);
        }
    }
}


// Phase 1, one m-column of one particle (compile-time M): monic q_l = ct q_{l-1} - gamma_lm q_{l-2}, q_M = st^M;
// rows of level l: q_l0 at l^2, (q_lM cos M phi, q_lM sin M phi) at l^2 + 2M - 1, l^2 + 2M.  Fy already points at
// the particle's element of (virtual) row 0; rows of levels outside [la, lb] are not stored.
template <int LMAX, int M, bool FULL>
__device__ __forceinline__ void acc_column(double ct, double st, const double* __restrict__ G, double* __restrict__ Fy,
                                           int la, int lb) {
    if constexpr (M <= LMAX) {
        double cm = 1.0, sm = 0.0, q1 = 1.0, q2 = 0.0;
        if (M > 0) { cm = G[(4 + M) * kAccP]; sm = G[(4 + kMaxL + M) * kAccP]; }
#pragma unroll
        for (int i = 0; i < M; ++i) q1 *= st;
#pragma unroll
        for (int l = M; l <= LMAX; ++l) {
            if (FULL || (l >= la && l <= lb)) {
                if (M == 0) Fy[(l * l) * kAccP] = q1;
                else { Fy[(l * l + 2 * M - 1) * kAccP] = q1 * cm; Fy[(l * l + 2 * M) * kAccP] = q1 * sm; }
            }
            if (l < LMAX) {
                const double qn = (l == M) ? ct * q1 : fma(ct, q1, -leg_gamma_c(l + 1, M) * q2);
                q2 = q1; q1 = qn;
            }
        }
    }
}

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// FULL: the table is a single unit group (la = 0, lb = LMAX): no per-row level tests in phase 1.
template <int LMAX, bool FULL>
__global__ void __launch_bounds__(kAccThreads, 1)
scf_accumulate_kernel(const double* __restrict__ pos, const double* __restrict__ mass, long long N,
                      const __grid_constant__ AccPlan pl, double* __restrict__ partial) {
    extern __shared__ __align__(16) double smem[];
    const AccGroup& g = pl.group[blockIdx.y];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* sG = smem;                                   // [2][kAccGRows][P]  geometry
    double* sX = sG + 2 * kAccGRows * kAccP;             // [2][4][P]          raw x, y, z, mass (cp.async landing zone)
    double* sF = sX + 2 * 4 * kAccP;                     // [2][nrows][P]      features
    const size_t fbuf = (size_t)g.nrows * kAccP;
    const int la = FULL ? 0 : g.la, lb = FULL ? LMAX : g.lb;

    // ---- roles -----------------------------------------------------------------------------------------
    const int my_unit = warp % g.nunits, my_rep = warp / g.nunits;
    const bool active = my_rep < g.rep;
    const AccUnit u = g.unit[my_unit];
    const int pk = tid & (kAccP - 1), pq = tid / kAccP;   // phase 1: particle, column class (0..3)

    double acc[kAccNCH][kAccWMax];
#pragma unroll
    for (int i = 0; i < kAccNCH; ++i)
#pragma unroll
        for (int j = 0; j < kAccWMax; ++j) acc[i][j] = 0.0;

    const int block = pl.block0 + (int)blockIdx.x;
    const long long pass0 = (long long)block * pl.passes_per_block;
    const long long pass1 = min(pl.passes, pass0 + pl.passes_per_block);

    // raw coordinates of a pass: global -> shared with cp.async, thread k moves (and later reads) element k only
    auto prefetch = [&](long long pass) {
        if (tid < kAccP && pass < pass1) {
            const long long k = pass * kAccP + tid;
            if (k < N) {
                double* X = sX + (size_t)(pass & 1) * 4 * kAccP + tid;
                cp_async8(X, pos + k);
                cp_async8(X + kAccP, pos + N + k);
                cp_async8(X + 2 * kAccP, pos + 2 * N + k);
                cp_async8(X + 3 * kAccP, mass + k);
            }
        }
    };
    auto phase0 = [&](long long pass) {
        if (tid < kAccP && pass < pass1) {
            cp_async_wait_all();
            double* G = sG + (size_t)(pass & 1) * kAccGRows * kAccP + tid;
            const double* X = sX + (size_t)(pass & 1) * 4 * kAccP + tid;
            const long long k = pass * kAccP + tid;
            double x = 1.0, y = 0.0, z = 0.0, mk = 0.0;   // padding particles carry zero mass
            if (k < N) { x = X[0]; y = X[kAccP]; z = X[2 * kAccP]; mk = X[3 * kAccP]; }
            const Geom gm = geometry(x, y, z);
            const double uu = __drcp_rn(1.0 + gm.r);
            G[0 * kAccP] = -uu * mk;               // m_k f_0,  f_l = -u s^l
            G[1 * kAccP] = (gm.r - 1.0) * uu;      // xi
            G[2 * kAccP] = gm.r * uu * uu;         // s
            G[3 * kAccP] = gm.ct;
            G[4 * kAccP] = gm.st;
            double cm = gm.cp, sm = gm.sp;
#pragma unroll
            for (int m = 1; m <= LMAX; ++m) {
                G[(4 + m) * kAccP] = cm;
                G[(4 + kMaxL + m) * kAccP] = sm;
                const double c2 = fma(cm, gm.cp, -sm * gm.sp);
                sm = fma(sm, gm.cp, cm * gm.sp);
                cm = c2;
            }
        }
    };
    auto phase1 = [&](long long pass) {
        if (pass >= pass1) return;
        const double* G = sG + (size_t)(pass & 1) * kAccGRows * kAccP + pk;
        double* F = sF + (size_t)(pass & 1) * fbuf + pk;
        double* Fy = F - (size_t)(la * la) * kAccP;   // row (l, f) of the group's buffer = l^2 + f - la^2
        const double ct = G[3 * kAccP], st = G[4 * kAccP];
        switch (pq) {   // warp-uniform: 4 warps per class
            case 0:
                acc_column<LMAX, 0, FULL>(ct, st, G, Fy, la, lb); acc_column<LMAX, 7, FULL>(ct, st, G, Fy, la, lb);
                acc_column<LMAX, 8, FULL>(ct, st, G, Fy, la, lb);
                break;
            case 1:
                acc_column<LMAX, 1, FULL>(ct, st, G, Fy, la, lb); acc_column<LMAX, 6, FULL>(ct, st, G, Fy, la, lb);
                acc_column<LMAX, 9, FULL>(ct, st, G, Fy, la, lb);
                break;
            case 2:
                acc_column<LMAX, 2, FULL>(ct, st, G, Fy, la, lb); acc_column<LMAX, 5, FULL>(ct, st, G, Fy, la, lb);
                acc_column<LMAX, 10, FULL>(ct, st, G, Fy, la, lb);
                break;
            default: {
                acc_column<LMAX, 3, FULL>(ct, st, G, Fy, la, lb); acc_column<LMAX, 4, FULL>(ct, st, G, Fy, la, lb);
                // radial seeds m_k f_l (rows after the Y rows) and xi
                const double sv = G[2 * kAccP];
                double f = G[0];
                double* Fs = F + (size_t)((lb + 1) * (lb + 1) - la * la - la) * kAccP;   // seed row of level l: Fs[l P]
#pragma unroll
                for (int l = 0; l <= LMAX; ++l) {
                    if (FULL || (l >= la && l <= lb)) Fs[l * kAccP] = f;
                    f *= sv;
                }
                Fs[(lb + 1) * kAccP] = G[1 * kAccP];
            }
        }
    };

    // ---- prologue: raw data of passes 0..2, geometry of passes 0 and 1, features of pass 0 ------------------
    prefetch(pass0);
    phase0(pass0);
    prefetch(pass0 + 1);
    phase0(pass0 + 1);
    prefetch(pass0 + 2);
    __syncthreads();
    phase1(pass0);
    __syncthreads();

    for (long long pass = pass0; pass < pass1; ++pass) {
        // Warps on one SM sub-partition (warp % 4) take the latency-bound feature phases and the FMA-bound accumulation in
        // opposite orders, so that the fp64 pipe has work while the other half waits on shared memory and rsqrt chains.
        const bool features_first = ((warp >> 2) & 1) == 0;
        phase0(pass + 2);     // writes G[pass&1] (last read by phase1(pass), before the previous barrier)
        prefetch(pass + 3);   // overwrites X[(pass+1)&1], consumed by this thread's phase0(pass+1) one iteration ago
        if (features_first) phase1(pass + 1);   // reads G[(pass+1)&1] (written before the previous barrier), writes F[(pass+1)&1]
        if (active) {         // reads F[pass&1] (written before the previous barrier)
            const double* F = sF + (size_t)(pass & 1) * fbuf;
            // single-group tables: code specialised per level (beta_n as immediates).  Multi-group tables run the generic
            // code for every unit: up to 11 levels x 4 widths of specialised code thrash the instruction cache
            // ((20,10), N = 1e7: 11.2 -> 9.5 ms with the generic path; (10,6) is the other way round, 132 vs 152 us)
            switch (u.w) {
                case 1: if (FULL) acc_unit_level<1>(F, g, u, g.rep, my_rep, lane, acc); else acc_unit_steps<1, -1>(F, g, u, g.rep, my_rep, lane, acc); break;
                case 2: if (FULL) acc_unit_level<2>(F, g, u, g.rep, my_rep, lane, acc); else acc_unit_steps<2, -1>(F, g, u, g.rep, my_rep, lane, acc); break;
                case 3: if (FULL) acc_unit_level<3>(F, g, u, g.rep, my_rep, lane, acc); else acc_unit_steps<3, -1>(F, g, u, g.rep, my_rep, lane, acc); break;
                default: if (FULL) acc_unit_level<4>(F, g, u, g.rep, my_rep, lane, acc); else acc_unit_steps<4, -1>(F, g, u, g.rep, my_rep, lane, acc); break;
            }
        }
        if (!features_first) phase1(pass + 1);
        __syncthreads();
    }

    // ---- lanes -> one value per accumulator (fixed butterfly), replicas in ascending order -----------------
#pragma unroll
    for (int i = 0; i < kAccNCH; ++i)
#pragma unroll
        for (int j = 0; j < kAccWMax; ++j) {
            double v = acc[i][j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            acc[i][j] = v;
        }
    if constexpr (FULL) {
        // Every lane now holds the warp's 44 totals.  Lane L hands on the entries a = L and a = L + 32 (a = i * kAccWMax + j): the
        // table index is computed once per lane instead of once per entry by lane 0 (ncu source view, N = 1e6: the write-out by
        // lane 0 — 44 guarded read-modify-writes and 44 stores with their index arithmetic — had 7 % of the kernel's samples).
        double mine[2] = {0.0, 0.0};
    #pragma unroll
        for (int i = 0; i < kAccNCH; ++i)
    #pragma unroll
            for (int j = 0; j < kAccWMax; ++j) {
                const int a = i * kAccWMax + j;
                if ((a & 31) == lane) mine[a >> 5] = acc[i][j];
            }
        int tix[2];
        bool ok[2];
    #pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int a = lane + 32 * h;
            const int i = a / kAccWMax, j = a % kAccWMax;
            const int n = u.n0 + i, f = u.f0 + j;
            const int m = (f + 1) >> 1;
            const bool is_sin = (f > 0) && ((f & 1) == 0);
            ok[h] = active && a < kAccNCH * kAccWMax && n < pl.n1 && j < u.w;
            tix[h] = ok[h] ? (is_sin ? pl.T : 0) + n * pl.L + lm_index(u.l, m) : 0;
        }
        double* sOut = smem;   // [2T]: cos table then sin table (entries of other groups stay untouched)
        __syncthreads();
        for (int r = 0; r < g.rep; ++r) {   // replicas of a unit are added in ascending order
            if (my_rep == r) {
    #pragma unroll
                for (int h = 0; h < 2; ++h)
                    if (ok[h]) sOut[tix[h]] = (r == 0) ? mine[h] : sOut[tix[h]] + mine[h];
            }
            __syncthreads();
        }
        if (my_rep == 0) {
            double* out = partial + (size_t)block * 2 * pl.T;
    #pragma unroll
            for (int h = 0; h < 2; ++h)
                if (ok[h]) out[tix[h]] = sOut[tix[h]];
        }
    } else {
        // multi-group tables (millions of particles per block pass loop: the write-out does not matter; with the compact form
        // ptxas moved spills into the pass loop of <10,false>: (20,10), N = 1e7, 9.72 -> 9.85 ms)
        double* sOut = smem;   // [2T]: cos table then sin table (entries of other groups stay untouched)
        __syncthreads();
        for (int r = 0; r < g.rep; ++r) {
            if (active && my_rep == r && lane == 0) {
    #pragma unroll
                for (int i = 0; i < kAccNCH; ++i)
    #pragma unroll
                    for (int j = 0; j < kAccWMax; ++j) {
                        const int n = u.n0 + i, f = u.f0 + j;
                        if (n < pl.n1 && j < u.w) {
                            const int m = (f + 1) >> 1;
                            const bool is_sin = (f > 0) && ((f & 1) == 0);
                            const int t = (is_sin ? pl.T : 0) + n * pl.L + lm_index(u.l, m);
                            sOut[t] = (r == 0) ? acc[i][j] : sOut[t] + acc[i][j];
                        }
                    }
            }
            __syncthreads();
        }
        if (active && my_rep == 0 && lane == 0) {
            double* out = partial + (size_t)block * 2 * pl.T;
    #pragma unroll
            for (int i = 0; i < kAccNCH; ++i)
    #pragma unroll
                for (int j = 0; j < kAccWMax; ++j) {
                    const int n = u.n0 + i, f = u.f0 + j;
                    if (n < pl.n1 && j < u.w) {
                        const int m = (f + 1) >> 1;
                        const bool is_sin = (f > 0) && ((f & 1) == 0);
                        const int t = (is_sin ? pl.T : 0) + n * pl.L + lm_index(u.l, m);
                        out[t] = sOut[t];
                    }
                }
        }
    }
}

// S5: fixed-order reduction over block partials and normalisation.  One warp per output: lane j sums the
// partials of blocks j, j+32, ... in ascending order, then a fixed butterfly combines the lanes.  The order
// depends only on `blocks` (a function of N and the table size), never on scheduling.
constexpr int kFinThreads = 256;

__global__ void __launch_bounds__(kFinThreads)
scf_finalize_kernel(const double* __restrict__ partial, int blocks, int nmax, int lmax,
                    double* __restrict__ A, double* __restrict__ B) {
    const int L = num_lm(lmax), T = (nmax + 1) * L;
    const int t = blockIdx.x * (kFinThreads / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (t >= 2 * T) return;
    const int tt = (t < T) ? t : t - T;
    const int n = tt / L, j = tt - n * L;
    int l = 0;
    while (lm_index(l + 1, 0) <= j) ++l;
    const int m = j - lm_index(l, 0);
    if (t >= T && m == 0) {   // B_{nl0}: no such feature was accumulated
        if (lane == 0) B[tt] = 0.0;
        return;
    }
    double s = 0.0;
    for (int b = lane; b < blocks; b += 32) s += partial[(size_t)b * 2 * T + t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane != 0) return;
    const double norm = (c_basis.norm_nl[l][n] * c_basis.geg_scale[l][n]) * (c_basis.N_lm[j] * c_basis.leg_scale[l][m]);
    if (t < T) A[tt] = norm * s;
    else B[tt] = norm * s;
}

// Sharded SCF (partial coefficients of every rank, then MPI_Allreduce): the tables of
// all ranks, gathered in rank order, are added in THAT order — the same bits on every rank and in every run.
__global__ void __launch_bounds__(256)
scf_combine_kernel(const double* __restrict__ parts, int nparts, long long len, double* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    double s = parts[i];
    for (int r = 1; r < nparts; ++r) s += parts[(size_t)r * len + i];
    out[i] = s;
}

cudaError_t scf_combine_launch(const double* parts, int nparts, long long len, double* out, cudaStream_t st) {
    scf_combine_kernel<<<(unsigned)((len + 255) / 256), 256, 0, st>>>(parts, nparts, len, out);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// Host side: plan, workspace, launches.
// ---------------------------------------------------------------------------------------------------------
constexpr int kAccMaxBlocksX = 148;

// Units in (level, n-chunk, feature tile) order; widths as equal as possible (2l+1 features in ceil(./4) tiles).
static AccPlan make_acc_plan(long long N, int nmax, int lmax) {
    AccPlan p{};
    p.nmax = nmax; p.lmax = lmax; p.n1 = nmax + 1; p.L = num_lm(lmax); p.T = p.n1 * p.L;
    const int nchunks = (p.n1 + kAccNCH - 1) / kAccNCH;
    AccUnit all[kAccMaxGroups * kAccWarps];
    int nu = 0;
    for (int l = 0; l <= lmax; ++l) {
        const int F = 2 * l + 1, tiles = (F + kAccWMax - 1) / kAccWMax;
        for (int c = 0; c < nchunks; ++c) {
            int f0 = 0;
            for (int t = 0; t < tiles; ++t) {
                const int w = F / tiles + (t < F % tiles ? 1 : 0);
                all[nu++] = AccUnit{(short)l, (short)f0, (short)w, (short)(c * kAccNCH)};
                f0 += w;
            }
        }
    }
    p.ngroups = (nu + kAccWarps - 1) / kAccWarps;
    for (int gi = 0; gi < p.ngroups; ++gi) {
        AccGroup& g = p.group[gi];
        // groups of (almost) equal size
        const int u0 = (int)((long long)nu * gi / p.ngroups), u1 = (int)((long long)nu * (gi + 1) / p.ngroups);
        g.nunits = u1 - u0;
        g.rep = kAccWarps / g.nunits;
        if (g.rep > kAccSteps) g.rep = kAccSteps;
        if (g.rep == 3) g.rep = 2;   // replicas take steps r, r+rep, ... of the 4 steps of a pass
        g.la = all[u0].l; g.lb = all[u1 - 1].l;
        // heavier units first is not needed: warp w sits on scheduler w % 4, and consecutive units have
        // similar widths, so every scheduler gets a similar sum of (W+2) * 11 operations
        for (int i = 0; i < g.nunits; ++i) g.unit[i] = all[u0 + i];
        g.nrows = (g.lb + 1) * (g.lb + 1) - g.la * g.la + (g.lb - g.la + 1) + 1;
    }
    p.passes = (N + kAccP - 1) / kAccP;
    long long bx = p.passes < kAccMaxBlocksX ? p.passes : kAccMaxBlocksX;
    p.passes_per_block = (p.passes + bx - 1) / bx;
    return p;
}

static int acc_blocks_x(const AccPlan& p) { return (int)((p.passes + p.passes_per_block - 1) / p.passes_per_block); }

static size_t acc_smem_bytes(const AccPlan& p) {
    int nrows = 0;
    for (int gi = 0; gi < p.ngroups; ++gi) nrows = p.group[gi].nrows > nrows ? p.group[gi].nrows : nrows;
    size_t b = (size_t)(2 * kAccGRows + 2 * 4 + 2 * nrows) * kAccP * sizeof(double);
    const size_t out = (size_t)2 * p.T * sizeof(double);
    return b > out ? b : out;
}

size_t scf_coeffs_workspace(long long N, int nmax, int lmax) {
    (void)N;
    return round_up((size_t)kAccMaxBlocksX * 2 * (nmax + 1) * num_lm(lmax) * sizeof(double), 256);
}

template <int LMAX>
static cudaError_t launch_accumulate(const double* pos, const double* mass, long long N, const AccPlan& p, int nblocks,
                                     double* partial, cudaStream_t st) {
    const size_t smem = acc_smem_bytes(p);
    if (p.ngroups == 1) scf_accumulate_kernel<LMAX, true><<<dim3(nblocks, 1), kAccThreads, smem, st>>>(pos, mass, N, p, partial);
    else scf_accumulate_kernel<LMAX, false><<<dim3(nblocks, p.ngroups), kAccThreads, smem, st>>>(pos, mass, N, p, partial);
    return cudaGetLastError();
}

// Blocks of the accumulation and the particles [first, last) block b works on: the host entry point uploads and
// accumulates ranges of whole blocks, which leaves every block partial — and so A, B — bit-identical to one launch.
int scf_coeffs_blocks(long long N, int nmax, int lmax, long long* particles_per_block) {
    const AccPlan p = make_acc_plan(N, nmax, lmax);
    if (particles_per_block) *particles_per_block = p.passes_per_block * kAccP;
    return acc_blocks_x(p);
}

cudaError_t scf_accumulate_launch(const double* pos, const double* mass, long long N, int nmax, int lmax, void* ws,
                                  int block0, int nblocks, cudaStream_t st) {
    cudaError_t e = scf_init_constants();
    if (e != cudaSuccess) return e;
    AccPlan p = make_acc_plan(N, nmax, lmax);
    p.block0 = block0;
    double* partial = static_cast<double*>(ws);
    switch (lmax) {
#define ETICS_CASE(LM) case LM: return launch_accumulate<LM>(pos, mass, N, p, nblocks, partial, st);
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5)
        ETICS_CASE(6) ETICS_CASE(7) ETICS_CASE(8) ETICS_CASE(9) ETICS_CASE(10)
#undef ETICS_CASE
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t scf_finalize_launch(long long N, int nmax, int lmax, double* A, double* B, const void* ws, cudaStream_t st) {
    const AccPlan p = make_acc_plan(N, nmax, lmax);
    const int T2 = 2 * p.T, wpb = kFinThreads / 32;
    scf_finalize_kernel<<<(T2 + wpb - 1) / wpb, kFinThreads, 0, st>>>(static_cast<const double*>(ws), acc_blocks_x(p), nmax, lmax, A, B);
    return cudaGetLastError();
}

cudaError_t scf_coeffs_launch(const double* pos, const double* mass, long long N, int nmax, int lmax,
                              double* A, double* B, void* ws, cudaStream_t st) {
    cudaError_t e = scf_accumulate_launch(pos, mass, N, nmax, lmax, ws, 0, scf_coeffs_blocks(N, nmax, lmax, nullptr), st);
    if (e != cudaSuccess) return e;
    return scf_finalize_launch(N, nmax, lmax, A, B, ws, st);
}

// nmax = 10 (the paper's cut-off) at lmax <= 6 gets fully unrolled n loops: 166.5 -> 149 us at N = 1e6.
// (20,10) with compile-time nmax and the n loops unrolled by 3: 6.41 -> 6.08 ms at N = 1e7 (fully unrolled — 5544
// FMAs of straight-line code — it was slower, 8.5 ms).
template <int LMAX>
constexpr int eval_n1c(int nmax) { return (LMAX <= 6 && nmax == 10) ? 11 : (LMAX == 10 && nmax == 20) ? 21 : 0; }

template <int LMAX, int N1C, bool PO>
static cudaError_t launch_eval_n(const double* pos, long long N, int nmax, const double* A, const double* B,
                                 double* acc, double* pot, cudaStream_t st) {
    constexpr int kEvalThreads = eval_threads(LMAX);
    const size_t smem = (size_t)(nmax + 1) * num_lm(LMAX) * sizeof(double2) + (size_t)(2 * LMAX + 2) * kEvalThreads * sizeof(double);
    long long blocks = (N + kEvalThreads - 1) / kEvalThreads;
    const long long cap = (long long)device_sm_count() * kEvalGridPerSM;
    if (eval_persistent(LMAX) && blocks > cap) blocks = cap;
    scf_eval_kernel<LMAX, N1C, PO><<<(unsigned)blocks, kEvalThreads, smem, st>>>(pos, N, nmax, A, B, acc, pot);
    return cudaGetLastError();
}

template <int LMAX, bool PO>
static cudaError_t launch_eval(const double* pos, long long N, int nmax, const double* A, const double* B,
                               double* acc, double* pot, cudaStream_t st) {
    if (LMAX <= 6 && nmax == 10) return launch_eval_n<LMAX, (LMAX <= 6 ? 11 : 0), PO>(pos, N, nmax, A, B, acc, pot, st);
    if (LMAX == 10 && nmax == 20) return launch_eval_n<LMAX, (LMAX == 10 ? 21 : 0), PO>(pos, N, nmax, A, B, acc, pot, st);
    return launch_eval_n<LMAX, 0, PO>(pos, N, nmax, A, B, acc, pot, st);
}

// what: ETICS_WHAT_BOTH | ETICS_WHAT_POTENTIAL (acc untouched) | ETICS_WHAT_FORCE (pot untouched)
cudaError_t scf_force_launch(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B, int what,
                             double* acc, double* pot, cudaStream_t st) {
    cudaError_t e = scf_init_constants();
    if (e != cudaSuccess) return e;
    if (what == ETICS_WHAT_FORCE) pot = nullptr;
    switch (lmax) {
#define ETICS_CASE(LM) case LM: return what == ETICS_WHAT_POTENTIAL ? launch_eval<LM, true>(pos, N, nmax, A, B, acc, pot, st) \
                                                                     : launch_eval<LM, false>(pos, N, nmax, A, B, acc, pot, st);
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5)
        ETICS_CASE(6) ETICS_CASE(7) ETICS_CASE(8) ETICS_CASE(9) ETICS_CASE(10)
#undef ETICS_CASE
        default: return cudaErrorInvalidValue;
    }
}

// ---- per-device set-up: constants and the dynamic shared-memory limit of every kernel instance, once per device ----------
constexpr int kMaxDynSmem = 227 * 1024;

template <int LM>
static cudaError_t set_kernel_attributes() {
    cudaError_t e = cudaSuccess;
    auto set = [&](auto kern) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
    };
    set(scf_accumulate_kernel<LM, true>);
    set(scf_accumulate_kernel<LM, false>);
    set(scf_eval_kernel<LM, 0, false>);
    set(scf_eval_kernel<LM, 0, true>);
    if constexpr (LM <= 6) { set(scf_eval_kernel<LM, 11, false>); set(scf_eval_kernel<LM, 11, true>); }
    if constexpr (LM == 10) { set(scf_eval_kernel<LM, 21, false>); set(scf_eval_kernel<LM, 21, true>); }
    if constexpr (LM > 0) { if (e == cudaSuccess) e = set_kernel_attributes<LM - 1>(); }
    return e;
}

cudaError_t scf_init_constants() {
    static DeviceOnce once;
    return once.run([] {
        cudaError_t e = etics_upload_constants_now();
        if (e != cudaSuccess) return e;
        {
            BasisConstants* c = new BasisConstants;
            fill_basis_constants(*c);
            auto* t = new double[2][kMaxL + 1][kMaxN + 1][kMaxL + 1];
            for (int l = 0; l <= kMaxL; ++l)
                for (int n = 0; n <= kMaxN; ++n)
                    for (int m = 0; m <= kMaxL; ++m) {
                        t[0][l][n][m] = c->leg_scale[l][m];
                        t[1][l][n][m] = c->geg_scale[l][n] * c->leg_scale[l][m];
                    }
            e = cudaMemcpyToSymbol(d_pack_scale, t, sizeof(double) * 2 * (kMaxL + 1) * (kMaxN + 1) * (kMaxL + 1));
            delete[] t;
            delete c;
            if (e != cudaSuccess) return e;
        }
        return set_kernel_attributes<kMaxL>();
    });
}

}  // namespace etics

// mex.cu — MEX half of the hot path (SURVEY.md §8(a) M1–M7) for sm_100a.
//
//   (mex_sort.cu)          M1-M2: keys = bits(r^2) (rounding pinned: t=x*x; t=fma(y,y,t); t=fma(z,z,t)), packed (x,y,z,m)
//                          records, stable radial sort -> permutation.
//   mex_gather_totals_kernel  M3+M4: sorted order -> per-particle geometry records (r, 1/r, cos/sin theta, cos/sin phi, m)
//                          in a chunk-transposed SoA layout that the scan kernels read fully coalesced; every lane
//                          owns K consecutive sorted particles, sums their moments m r^l P_lm {cos,sin} m phi and
//                          m r^-(l+1) P_lm {cos,sin} m phi, and the warp adds the 32 chunk sums: tile totals.
//   mex_tilescan_kernel    M5b: exclusive scan of the tile totals (forward for q, backward for p), fixed order.
//   mex_evaluate_kernel    M5a+M5c+M6+M7: each lane recomputes its chunk sums, the warp scans them in shared memory
//                          (inside-out for q, outside-in for p), then each lane re-walks its K particles forwards
//                          carrying q and backwards carrying p (never "total minus prefix": that cancels
//                          catastrophically), accumulates potential and spherical force components, transforms
//                          to Cartesian and scatters one 32-byte record to the particle's original index.
//   mex_unpack_kernel      records -> acc (3,N), pot (N).
//
// The fp64 scans use a fixed summation order (thread chunk -> tile -> grid), so results are bitwise reproducible.
// The (l,m) set is split into groups of whole m-columns (the Legendre l-recurrence runs along a column), so a
// thread never holds more than 28 running sums per direction in registers at a time.
//
// What the paper did instead (prior art, §3.2): Thrust merge sort of particle structs, a cache
// kernel, then per l: a summand kernel writing q_lm, p_lm of every particle to global memory, one Thrust
// exclusive_scan per (m, re/im, direction), a partial-force kernel; finally a coordinate-transform kernel.
#include "mex_common.cuh"

// This file is compiled four times (paper_1406_4254_b200/build.py) with ETICS_MEX_PART = 0..3: part 0 holds the workspace
// layout, the host entry points and the scan kernels for lmax <= 6; parts 1-3 only instantiate the scan kernels for lmax 7-8, 9
// and 10 — the template instances dominate the compile time and the parts build in parallel.
#ifndef ETICS_MEX_PART
#define ETICS_MEX_PART 0
#endif

namespace etics {

#if ETICS_MEX_PART == 0
int mex_kernel_launches(long long N) { return mex_sort_kernel_launches(N) + 4; }   // + gather/totals, tile scan, evaluate, unpack
cudaError_t mex_init_constants() { return mex_sort_init_device(); }   // every MEX constant is a compile-time literal; per-device function attributes
#endif

// =========================================================================================================
// Column groups.  Column m holds the pairs (l,m), l = m..LMAX; a group is a set of whole columns.
// =========================================================================================================
// Column -> group tables: greedy balanced partition (columns in descending count of running sums, each to the least
// loaded group) for a target of 28 running sums per direction and group; generated offline, fixed at compile time.
// (Targets of 17 and 13 sums per group — 3 and 4 groups at lmax 6, 128 registers, 16 resident warps per SM instead of 12 —
// were measured again with the fused kernel: 125 -> 139 and 154 us at N = 1e6: every group repeats the per-particle set-up.)
constexpr int kMexMaxGroups = 8;

#define ETICS_MEX_NG_INIT {1, 1, 1, 1, 1, 2, 2, 3, 3, 4, 5}
#define ETICS_MEX_GOF_INIT { \
    {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, \
    {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, \
    {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, \
    {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, \
    {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, \
    {1, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0}, \
    {0, 0, 1, 1, 1, 0, 0, 0, 0, 0, 0}, \
    {2, 0, 1, 2, 1, 0, 2, 0, 0, 0, 0}, \
    {1, 0, 1, 2, 2, 0, 2, 1, 0, 0, 0}, \
    {3, 0, 1, 2, 3, 2, 1, 0, 3, 0, 0}, \
    {4, 0, 1, 2, 3, 4, 3, 2, 1, 0, 4}}
__host__ __device__ constexpr int mex_num_groups(int lmax) {
    constexpr int t[ETICS_MAX_LMAX + 1] = ETICS_MEX_NG_INIT;
    return t[lmax];
}
__host__ __device__ constexpr int mex_group_of(int lmax, int m) {
    constexpr int t[ETICS_MAX_LMAX + 1][ETICS_MAX_LMAX + 1] = ETICS_MEX_GOF_INIT;
    return t[lmax][m];
}
// running sums per direction of column m: cos only for m = 0, (cos, sin) otherwise
__host__ __device__ constexpr int mex_col_slots(int lmax, int m) { return (lmax - m + 1) * (m == 0 ? 1 : 2); }
// first slot of column m inside its group
__host__ __device__ constexpr int mex_slot_base(int lmax, int m) {
    int s = 0;
    for (int mm = 0; mm < m; ++mm)
        if (mex_group_of(lmax, mm) == mex_group_of(lmax, m)) s += mex_col_slots(lmax, mm);
    return s;
}
__host__ __device__ constexpr int mex_group_slots(int lmax, int g) {
    int s = 0;
    for (int m = 0; m <= lmax; ++m)
        if (mex_group_of(lmax, m) == g) s += mex_col_slots(lmax, m);
    return s;
}
// first global row of group g; rows of a group: [0,NS) = q slots (forward), [NS,2NS) = p slots (backward)
__host__ __device__ constexpr int mex_row_base(int lmax, int g) {
    int s = 0;
    for (int gg = 0; gg < g; ++gg) s += 2 * mex_group_slots(lmax, gg);
    return s;
}
__host__ __device__ constexpr int mex_total_rows(int lmax) { return mex_row_base(lmax, mex_num_groups(lmax)); }
__host__ __device__ constexpr int mex_max_group_slots(int lmax) {
    int s = 0;
    for (int g = 0; g < mex_num_groups(lmax); ++g) s = mex_group_slots(lmax, g) > s ? mex_group_slots(lmax, g) : s;
    return s;
}
// w_lm = (2 - delta_m0) (l-m)!/(l+m)!   (eq. 15's 4 pi/(2l+1) times the orthonormal Y_lm normalisation, +-m folded)
__host__ __device__ constexpr double mex_w(int l, int m) {
    double v = (m == 0) ? 1.0 : 2.0;
    for (int k = l - m + 1; k <= l + m; ++k) v /= double(k);
    return v;
}
__host__ __device__ constexpr double mex_dfact(int m) {   // (2m-1)!!
    double v = 1.0;
    for (int k = 1; k <= m; ++k) v *= double(2 * k - 1);
    return v;
}

#if ETICS_MEX_PART == 0
MexLayout make_mex_layout(long long N, int lmax) {
    MexLayout L{};
    L.N = N; L.lmax = lmax;
    L.tiles = (N + kMexTile - 1) / kMexTile;
    L.chunks = L.tiles * kMexThreads;
    L.rows = mex_total_rows(lmax);
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += round_up(bytes, 256); return at; };
    L.off_hdr = take(sizeof(SortHeader));
    L.off_seghist = take((size_t)kSortMaxSegs * kSortBins * sizeof(unsigned));
    L.off_bintot = take((size_t)kSortBins * sizeof(unsigned));
    L.off_keys = take((size_t)N * 8);
    L.off_wordsA = take((size_t)N * 8);
    L.off_wordsB = take((size_t)N * 8);
    L.off_perm = take((size_t)N * 4);
    L.off_itmp = take((size_t)N * 4);
    L.off_pk = take((size_t)N * 32);
    L.off_rec = take((size_t)L.tiles * kRecFields * kMexTile * 8);
    L.off_idxT = take((size_t)L.tiles * kMexTile * 4);
    L.off_tot = take((size_t)L.rows * L.tiles * 8);
    L.total = o;
    return L;
}

size_t mex_workspace(long long N, int lmax) { return make_mex_layout(N, lmax).total; }
#endif

// =========================================================================================================
// M3: gather into geometry records.  Record of the particle at sorted position p = tile*TP + c*K + k
// (chunk c, step k) is stored field by field at rec[tile][field][k][c], so that the threads of the scan
// kernels (thread = chunk c) read consecutive doubles.  Padding positions (p >= N) get a massless particle.
// =========================================================================================================
struct Rec { double r, rinv, ct, st, cp, sp, mass; };

__device__ __forceinline__ Rec load_rec(const double* __restrict__ rec_tile, int k, int c) {
    const double* b = rec_tile + k * kMexThreads + c;
    Rec p;
    p.r = b[0 * kMexTile]; p.rinv = b[1 * kMexTile]; p.ct = b[2 * kMexTile]; p.st = b[3 * kMexTile];
    p.cp = b[4 * kMexTile]; p.sp = b[5 * kMexTile]; p.mass = b[6 * kMexTile];
    return p;
}

__device__ __forceinline__ Rec load_rec_cg(const double* rec_tile, int k, int c) {   // records written earlier by this kernel
    const double* b = rec_tile + k * kMexThreads + c;
    Rec p;
    p.r = __ldcg(b + 0 * kMexTile); p.rinv = __ldcg(b + 1 * kMexTile); p.ct = __ldcg(b + 2 * kMexTile); p.st = __ldcg(b + 3 * kMexTile);
    p.cp = __ldcg(b + 4 * kMexTile); p.sp = __ldcg(b + 5 * kMexTile); p.mass = __ldcg(b + 6 * kMexTile);
    return p;
}

// =========================================================================================================
// Per-particle column arithmetic (eqs. 15–17; real form and weights: DESIGN.md "Readings").
// Column m, stable l-recurrence (never the paper's eq. 24), in MONIC form so that every step
// is one multiply and one FMA:
//   P_lm = h_lm sin(theta) u_lm (m >= 1),  P_l0 = h_l0 u_l0;   h_mm = (2m-1)!!,  h_lm = h_{l-1,m} (2l-1)/(l-m)
//   u_mm = st^(m-1) (u_00 = 1),  u_{m+1,m} = ct u_mm,  u_lm = ct u_{l-1,m} - gamma_lm u_{l-2,m},
//   gamma_lm = (l+m-1)(l-1-m) / ((2l-1)(2l-3))
// (u_lm sin(theta) = P_lm / h_lm; u_lm itself is a polynomial in ct, st: nothing is divided by sin theta.)
// The running sums carry the weight W_lm = w_lm h_lm^2 (one P from the source particle, one from the target):
//   S^{c,s}_lm = sum_j W_lm m_j {r_j^l | r_j^-(l+1)} Y_lm(j) {cos, sin}(m phi_j),   Y_lm = st u_lm  (Y_l0 = u_l0)
// Same-column derivative: (dP_lm/dtheta)/h_lm = l ct u_lm - (l+m)(l-m)/(2l-1) u_{l-1,m}  (m >= 1);
//                         (dP_l0/dtheta)/h_l0 = -l st u_l1   (h_l1 / h_l0 = l).
// =========================================================================================================
__host__ __device__ constexpr double mex_h(int l, int m) {
    double v = mex_dfact(m);
    for (int k = m + 1; k <= l; ++k) v = v * double(2 * k - 1) / double(k - m);
    return v;
}
__host__ __device__ constexpr double mex_W(int l, int m) { return mex_w(l, m) * mex_h(l, m) * mex_h(l, m); }
__host__ __device__ constexpr double mex_gamma(int l, int m) {
    return (l >= m + 2) ? double((l + m - 1) * (l - 1 - m)) / double((2 * l - 1) * (2 * l - 3)) : 0.0;
}
__host__ __device__ constexpr bool mex_in_group(int lmax, int g, int m) { return m <= lmax && mex_group_of(lmax, m) == g; }

// cos(m phi), sin(m phi), st^(m-1) of the columns of group G (the chains run over every m; unused entries vanish)
template <int LMAX>
struct Angles {
    double cm[LMAX + 1], sm[LMAX + 1];   // cos m phi, sin m phi
    double sp1[LMAX + 1];                // st^(m-1), m >= 1
    __device__ __forceinline__ void init(const Rec& p) {
        // cos(m phi), sin(m phi) by the three-term recurrence f_m = 2 cos(phi) f_{m-1} - f_{m-2}: one FMA per value
        cm[0] = 1.0; sm[0] = 0.0; sp1[0] = 0.0;
        const double tc = p.cp + p.cp;
#pragma unroll
        for (int m = 1; m <= LMAX; ++m) {
            cm[m] = (m == 1) ? p.cp : fma(tc, cm[m - 1], -cm[m - 2]);
            sm[m] = (m == 1) ? p.sp : fma(tc, sm[m - 1], -sm[m - 2]);
            sp1[m] = (m == 1) ? 1.0 : sp1[m - 1] * p.st;
        }
    }
};

// moments of one particle into the UNWEIGHTED chunk sums of group G (both directions): q[], pq[] have NS entries.
// m >= 1: sum of (m r^l st) u_lm {cos, sin} m phi;  m = 0: sum of (m r^l) u_l0.  mex_weight_sums applies W_lm once per chunk.
template <int LMAX, int G>
__device__ __forceinline__ void mex_agg_particle(const Rec& p, double* __restrict__ q, double* __restrict__ pq) {
    Angles<LMAX> a;
    a.init(p);
    double mq[LMAX + 1], mp[LMAX + 1];   // m r^l, m r^-(l+1)
    mq[0] = p.mass; mp[0] = p.mass * p.rinv;
#pragma unroll
    for (int l = 1; l <= LMAX; ++l) { mq[l] = mq[l - 1] * p.r; mp[l] = mp[l - 1] * p.rinv; }
#pragma unroll
    for (int m = 0; m <= LMAX; ++m) {
        if (!mex_in_group(LMAX, G, m)) continue;
        const int sb = mex_slot_base(LMAX, m);
        double u1 = 0.0, u2 = 0.0;   // u_{l-1,m}, u_{l-2,m}
#pragma unroll
        for (int l = m; l <= LMAX; ++l) {
            double u;
            if (l == m) u = (m == 0) ? 1.0 : a.sp1[m] * p.st;   // m >= 1: the chain carries st u_lm = Y_lm
            else if (l == m + 1) u = p.ct * u1;
            else u = fma(p.ct, u1, -mex_gamma(l, m) * u2);
            u2 = u1; u1 = u;
            if (m == 0) {
                q[sb + l] = fma(mq[l], u, q[sb + l]);
                pq[sb + l] = fma(mp[l], u, pq[sb + l]);
            } else {
                const double tq = mq[l] * u, tp = mp[l] * u;
                const int s = sb + 2 * (l - m);
                q[s] = fma(tq, a.cm[m], q[s]);       q[s + 1] = fma(tq, a.sm[m], q[s + 1]);
                pq[s] = fma(tp, a.cm[m], pq[s]);     pq[s + 1] = fma(tp, a.sm[m], pq[s + 1]);
            }
        }
    }
}

template <int LMAX, int G>
__device__ __forceinline__ void mex_weight_sums(double* __restrict__ q, double* __restrict__ pq) {
#pragma unroll
    for (int m = 0; m <= LMAX; ++m) {
        if (!mex_in_group(LMAX, G, m)) continue;
        const int sb = mex_slot_base(LMAX, m);
#pragma unroll
        for (int l = m; l <= LMAX; ++l) {
            if (m == 0) {
                q[sb + l] *= mex_W(l, 0); pq[sb + l] *= mex_W(l, 0);
            } else {
                const int s = sb + 2 * (l - m);
                q[s] *= mex_W(l, m); q[s + 1] *= mex_W(l, m); pq[s] *= mex_W(l, m); pq[s + 1] *= mex_W(l, m);
            }
        }
    }
}

// Evaluate the group-G part of (Phi, a_r, a_theta, a_phi) at one particle from the running sums s[] of one
// direction, THEN add the particle's own moment (exclusive sums, eqs. 11–12).
//   FWD: s = q (interior), radial factor r^-(l+1), d/dr factor -(l+1)/r;  own moment m r^l
//   BWD: s = p (exterior), radial factor r^l,      d/dr factor  l/r;      own moment m r^-(l+1)
// Level by level: the m sums of a level (P, dP/dtheta, U-weighted) are formed first and meet the radial factor
// once per level.  out[0..3] += (Phi, a_r, a_theta, a_phi) contributions.
// PO: potential only: the derivative sums are not formed.
template <int LMAX, int G, bool FWD, bool PO>
__device__ __forceinline__ void mex_eval_particle(const Rec& p, double* __restrict__ s, double* __restrict__ out) {
    Angles<LMAX> a;
    a.init(p);
    double mcm[LMAX + 1], msm[LMAX + 1];   // m cos(m phi), m sin(m phi): the d/dphi factor rides on the rotation
#pragma unroll
    for (int m = 1; m <= LMAX; ++m) { mcm[m] = double(m) * a.cm[m]; msm[m] = double(m) * a.sm[m]; }
    constexpr bool kAux1 = mex_in_group(LMAX, G, 0) && !mex_in_group(LMAX, G, 1) && LMAX >= 1;   // m = 0 needs u_l1
    double u1[LMAX + 1], u2[LMAX + 1];     // u_{l-1,m}, u_{l-2,m} per column
#pragma unroll
    for (int m = 0; m <= LMAX; ++m) { u1[m] = 0.0; u2[m] = 0.0; }
    double x1 = 0.0, x2 = 0.0;             // the auxiliary m = 1 column when it lives in another group
    double rho = FWD ? p.rinv : 1.0;       // r^-(l+1) | r^l
    double mu = FWD ? p.mass : p.mass * p.rinv;   // m r^l | m r^-(l+1)
    double sP = 0.0, sR = 0.0, sT = 0.0, sF = 0.0;
#pragma unroll
    for (int l = 0; l <= LMAX; ++l) {
        // ---- the level's u_lm ---------------------------------------------------------------------------
        double u[LMAX + 1];
#pragma unroll
        for (int m = 0; m <= l; ++m) {
            if (!mex_in_group(LMAX, G, m)) continue;
            if (l == m) u[m] = (m == 0) ? 1.0 : a.sp1[m];
            else if (l == m + 1) u[m] = p.ct * u1[m];
            else u[m] = fma(p.ct, u1[m], -mex_gamma(l, m) * u2[m]);
        }
        double ul1 = 0.0;                  // u_l1, for dP_l0/dtheta
        if (mex_in_group(LMAX, G, 0) && l >= 1) {
            if (kAux1) {
                const double x = (l == 1) ? 1.0 : (l == 2) ? p.ct * x1 : fma(p.ct, x1, -mex_gamma(l, 1) * x2);
                x2 = x1; x1 = x;
                ul1 = x;
            } else {
                ul1 = u[1];
            }
        }
        // ---- sums over the group's m at this level, then the own moment ------------------------------------
        //   sum_m P_lm E_m          = u_l0 E_0 + st aU,                 aU = sum_{m>=1} u_lm E_m
        //   sum_m (dP_lm/dth) E_m   = -l st u_l1 E_0 + l ct aU - aV,    aV = sum_{m>=1, m<l} c_lm u_{l-1,m} E_m
        //   sum_m m U_lm F'_m       = aF                                 (all in units of h_lm; W_lm rides on the sums)
        const double mus = mu * p.st;
        double aU = 0.0, aV = 0.0, aF = 0.0, aP0 = 0.0, aT0 = 0.0;
#pragma unroll
        for (int m = 0; m <= l; ++m) {
            if (!mex_in_group(LMAX, G, m)) continue;
            const int sb = mex_slot_base(LMAX, m);
            if (m == 0) {
                const double e = s[sb + l];
                aP0 = u[0] * e;
                if (!PO && l >= 1) aT0 = (-(double(l) * p.st) * ul1) * e;
                s[sb + l] = fma(mex_W(l, 0) * mu, u[0], e);
            } else {
                const int i = sb + 2 * (l - m);
                const double E = fma(s[i], a.cm[m], s[i + 1] * a.sm[m]);
                aU = fma(u[m], E, aU);
                if (!PO) aF = fma(u[m], fma(s[i + 1], mcm[m], -s[i] * msm[m]), aF);
                if (!PO && m < l) aV = fma((double((l + m) * (l - m)) / double(2 * l - 1)) * u1[m], E, aV);
                const double t = (mex_W(l, m) * mus) * u[m];
                s[i] = fma(t, a.cm[m], s[i]);
                s[i + 1] = fma(t, a.sm[m], s[i + 1]);
            }
        }
        const double aP = fma(p.st, aU, aP0);
        const double pa = rho * aP;
        sP += pa;
        if (!PO) {
            const double aT = fma(double(l) * p.ct, aU, aT0 - aV);
            sR = fma(FWD ? -double(l + 1) : double(l), pa, sR);
            sT = fma(rho, aT, sT);
            sF = fma(rho, aF, sF);
        }
        rho *= FWD ? p.rinv : p.r;
        mu *= FWD ? p.r : p.rinv;
#pragma unroll
        for (int m = 0; m <= l; ++m)
            if (mex_in_group(LMAX, G, m)) { u2[m] = u1[m]; u1[m] = u[m]; }
    }
    out[0] -= sP;
    if (!PO) {
        out[1] = fma(p.rinv, sR, out[1]);
        out[2] = fma(p.rinv, sT, out[2]);
        out[3] = fma(p.rinv, sF, out[3]);
    }
}

// =========================================================================================================
// M3 + M4: gather into geometry records and tile totals of the moments.  A tile is ONE WARP: lane = chunk of kMexK
// consecutive sorted particles (no block barrier anywhere).
//   1. the lane reads its 8 permutation entries (32 contiguous bytes) and the 8 packed (x,y,z,m) sectors, computes the
//      geometry and stores the records (field-major, chunk-transposed: coalesced) and the indices;
//   2. per column group the lane sums the moments of its chunk in registers (records re-read through L2 for the
//      groups after the first);
//   3. the sums go to shared memory transposed (V[row][33]) and lane = row adds the 32 chunk sums in chunk order:
//      tot[row][tile].  The chunk sums themselves are NOT stored: the evaluation kernel recomputes them (98-180 bytes
//      per particle written and read back in round 1).
// =========================================================================================================
constexpr int kVStride = kMexThreads + 1;
static_assert(kMexThreads == 32, "the MEX scan kernels use warp-sized tiles");

// CG: the records were written earlier by the calling kernel (read them through L2, not the non-coherent path)
template <int LMAX, int G, bool CG>
__device__ __forceinline__ void mex_chunk_sums(const double* rec_tile, int c, double* __restrict__ q, double* __restrict__ pq) {
    constexpr int NS = mex_group_slots(LMAX, G);
#pragma unroll
    for (int s = 0; s < NS; ++s) { q[s] = 0.0; pq[s] = 0.0; }
    // the next record (lmax >= 7: the next two) is loaded while the current one is processed: a particle's moments are 270-450
    // fp64 operations, about an L2 round trip with three warps per scheduler (two ahead at lmax 6 costs registers: spills)
    auto ld = [&](int k) { return CG ? load_rec_cg(rec_tile, k < kMexK ? k : kMexK - 1, c) : load_rec(rec_tile, k < kMexK ? k : kMexK - 1, c); };
    if constexpr (LMAX >= 7) {
        Rec p = ld(0), n1 = ld(1);
#pragma unroll 2
        for (int k = 0; k < kMexK; ++k) {
            const Rec n2 = ld(k + 2);
            mex_agg_particle<LMAX, G>(p, q, pq);
            p = n1; n1 = n2;
        }
    } else {
        Rec p = ld(0);
#pragma unroll 1
        for (int k = 0; k < kMexK; ++k) {
            const Rec n1 = ld(k + 1);
            mex_agg_particle<LMAX, G>(p, q, pq);
            p = n1;
        }
    }
    mex_weight_sums<LMAX, G>(q, pq);
}

template <int LMAX, int G>
__device__ __forceinline__ void mex_totals_group(const double* rec_tile, double* V, double* __restrict__ tot,
                                                 long long tiles, long long tile) {
    constexpr int NS = mex_group_slots(LMAX, G);
    constexpr int RB = mex_row_base(LMAX, G);
    constexpr int ROWS = 2 * NS;
    const int c = threadIdx.x;
    double q[NS], pq[NS];
    mex_chunk_sums<LMAX, G, true>(rec_tile, c, q, pq);
#pragma unroll
    for (int s = 0; s < NS; ++s) { V[s * kVStride + c] = q[s]; V[(NS + s) * kVStride + c] = pq[s]; }
    __syncwarp();
    for (int row = c; row < ROWS; row += kMexThreads) {
        const double* v = V + row * kVStride;
        // four interleaved partial sums (chunks j = 0, 4, 8, ...; 1, 5, ...; ...), then a fixed tree: a quarter of the
        // dependent-add chain of a serial row sum, the same order in every run
        double r0 = 0.0, r1 = 0.0, r2 = 0.0, r3 = 0.0;
#pragma unroll
        for (int j = 0; j < kMexThreads; j += 4) { r0 += v[j]; r1 += v[j + 1]; r2 += v[j + 2]; r3 += v[j + 3]; }
        tot[(size_t)(RB + row) * tiles + tile] = (r0 + r1) + (r2 + r3);
    }
    __syncwarp();
}

template <int LMAX>
__global__ void __launch_bounds__(kMexThreads)
mex_gather_totals_kernel(const double2* __restrict__ pk, const unsigned* __restrict__ perm, long long N, long long tiles,
                         double* rec, unsigned* __restrict__ idxT, double* __restrict__ tot) {
    constexpr int MAXROWS = 2 * mex_max_group_slots(LMAX);
    __shared__ double V[MAXROWS * kVStride];
    const long long tile = blockIdx.x;
    const int c = threadIdx.x;
    double* rec_tile = rec + (size_t)tile * kRecFields * kMexTile;
    const long long p0 = tile * kMexTile + (long long)c * kMexK;
    unsigned idx[kMexK];
    if (p0 + kMexK <= N) {
        static_assert(kMexK % 4 == 0, "the permutation entries of a chunk are read as 16-byte vectors");
#pragma unroll
        for (int k = 0; k < kMexK; k += 4) {
            const uint4 a = *reinterpret_cast<const uint4*>(perm + p0 + k);
            idx[k] = a.x; idx[k + 1] = a.y; idx[k + 2] = a.z; idx[k + 3] = a.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < kMexK; ++k) idx[k] = (p0 + k < N) ? perm[p0 + k] : 0xffffffffu;
    }
    double2 xy[kMexK], zm[kMexK];
#pragma unroll
    for (int k = 0; k < kMexK; ++k) {
        const bool ok = p0 + k < N;
        xy[k] = make_double2(1.0, 0.0); zm[k] = make_double2(0.0, 0.0);       // padding: a massless particle
        if (ok)   // the 32-byte record in ONE load (two 16-byte loads of the same sector: 4.75 -> 4.71 ms at N = 1e8)
            asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];"
                         : "=d"(xy[k].x), "=d"(xy[k].y), "=d"(zm[k].x), "=d"(zm[k].y) : "l"(pk + 2 * (size_t)idx[k]));
    }
#pragma unroll
    for (int k = 0; k < kMexK; ++k) {
        const Geom g = geometry(xy[k].x, xy[k].y, zm[k].x);
        double* b = rec_tile + k * kMexThreads + c;
        b[0 * kMexTile] = g.r; b[1 * kMexTile] = g.rinv; b[2 * kMexTile] = g.ct; b[3 * kMexTile] = g.st;
        b[4 * kMexTile] = g.cp; b[5 * kMexTile] = g.sp; b[6 * kMexTile] = zm[k].y;
        idxT[(size_t)tile * kMexTile + k * kMexThreads + c] = (p0 + k < N) ? idx[k] : 0u;
    }
    constexpr int NG = mex_num_groups(LMAX);
    mex_totals_group<LMAX, 0>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 1) mex_totals_group<LMAX, 1>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 2) mex_totals_group<LMAX, 2>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 3) mex_totals_group<LMAX, 3>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 4) mex_totals_group<LMAX, 4>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 5) mex_totals_group<LMAX, 5>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 6) mex_totals_group<LMAX, 6>(rec_tile, V, tot, tiles, tile);
    if constexpr (NG > 7) mex_totals_group<LMAX, 7>(rec_tile, V, tot, tiles, tile);
}

// =========================================================================================================
// M5b: exclusive scan of the tile totals tot[row][tile], one block per row, fixed order.  Rows [rb, rb+ns) of a
// group run forward (q), rows [rb+ns, rb+2ns) backward (p).  256 tiles per step: coalesced load, warp-shuffle
// scan, carry to the next step.
// =========================================================================================================
struct RowDirs { int ng; int rb[kMexMaxGroups]; int ns[kMexMaxGroups]; };
constexpr int kTileScanThreads = 256;   // 1024 threads (8192 tiles per step) were slower: 14.7 -> 20.9 us at N = 1e6, 0.60 -> 0.79 ms at 1e8 (lmax 8)
constexpr int kTileScanItems = 8;   // consecutive scan-order positions per thread and step

static __global__ void __launch_bounds__(kTileScanThreads)
mex_tilescan_kernel(double* __restrict__ tot, long long tiles, RowDirs rd, const double* __restrict__ base) {
    __shared__ double wsum[kTileScanThreads / 32];
    const int row = blockIdx.x, t = threadIdx.x, lane = t & 31, warp = t >> 5;
    bool fwd = true;
    for (int g = 0; g < rd.ng; ++g)
        if (row >= rd.rb[g] && row < rd.rb[g] + 2 * rd.ns[g]) fwd = row < rd.rb[g] + rd.ns[g];
    double* v = tot + (size_t)row * tiles;
    // radius-partitioned MEX: the scan starts from the sums of the shards inside (q rows) / outside (p rows) this one
    double carry = base ? base[row] : 0.0;
    for (long long b0 = 0; b0 < tiles; b0 += kTileScanThreads * kTileScanItems) {
        const long long j0 = b0 + (long long)t * kTileScanItems;   // first scan-order position of this thread
        double x[kTileScanItems];
#pragma unroll
        for (int e = 0; e < kTileScanItems; ++e) {
            const long long j = j0 + e;
            x[e] = (j < tiles) ? v[fwd ? j : tiles - 1 - j] : 0.0;
        }
        double local = 0.0;
#pragma unroll
        for (int e = 0; e < kTileScanItems; ++e) local += x[e];
        double inc = local;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        if (lane == 31) wsum[warp] = inc;
        double exc = __shfl_up_sync(0xffffffffu, inc, 1);
        if (lane == 0) exc = 0.0;
        __syncthreads();
        double woff = 0.0, total = 0.0;
#pragma unroll
        for (int w = 0; w < kTileScanThreads / 32; ++w) {
            const double s = wsum[w];
            if (w < warp) woff += s;
            total += s;
        }
        __syncthreads();
        double run = carry + (woff + exc);
#pragma unroll
        for (int e = 0; e < kTileScanItems; ++e) {
            const long long j = j0 + e;
            if (j < tiles) v[fwd ? j : tiles - 1 - j] = run;
            run += x[e];
        }
        carry += total;
    }
}

// Radius-partitioned MEX: the sum of every row of the tile totals = this shard's moment
// vector.  One block per row; thread t adds the tiles t, t + 256, ... in order, then a fixed tree over the threads.
static __global__ void __launch_bounds__(kTileScanThreads)
mex_rowtotal_kernel(const double* __restrict__ tot, long long tiles, double* __restrict__ totals) {
    __shared__ double part[kTileScanThreads];
    const int row = blockIdx.x, t = threadIdx.x;
    const double* v = tot + (size_t)row * tiles;
    double s = 0.0;
    for (long long j = t; j < tiles; j += kTileScanThreads) s += v[j];
    part[t] = s;
    __syncthreads();
    for (int o = kTileScanThreads / 2; o > 0; o >>= 1) {
        if (t < o) part[t] += part[t + o];
        __syncthreads();
    }
    if (t == 0) totals[row] = part[0];
}

#if ETICS_MEX_PART == 0
// base[row] of shard `rank` from the shards' moment vectors parts[s][row], s in radius order: q rows (inside-out) take the
// shards inside, added from the innermost outwards; p rows (outside-in) the shards outside, added from the outermost inwards.
static __global__ void mex_shard_bases_kernel(const double* __restrict__ parts, int nparts, int rank, int rows, RowDirs rd,
                                              double* __restrict__ base) {
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= rows) return;
    bool fwd = true;
    for (int g = 0; g < rd.ng; ++g)
        if (row >= rd.rb[g] && row < rd.rb[g] + 2 * rd.ns[g]) fwd = row < rd.rb[g] + rd.ns[g];
    double s = 0.0;
    if (fwd) for (int k = 0; k < rank; ++k) s += parts[(size_t)k * rows + row];
    else for (int k = nparts - 1; k > rank; --k) s += parts[(size_t)k * rows + row];
    base[row] = s;
}
#endif

// =========================================================================================================
// M5c + M6 + M7: walk, evaluate, transform, scatter.
// Shared memory: out[k][4][lane] (Phi, a_r, a_theta, a_phi of the lane's K particles; lane-private columns).
// =========================================================================================================
template <int LMAX, int G, bool PO>
__device__ __forceinline__ void mex_evaluate_group(const double* __restrict__ rec_tile, double* sOut, double* V,
                                                   const double* __restrict__ tot, long long tiles, long long tile) {
    constexpr int NS = mex_group_slots(LMAX, G);
    constexpr int RB = mex_row_base(LMAX, G);
    static_assert(NS <= kMexThreads, "one lane per row in the chunk scan");
    const int c = threadIdx.x;
    double s[NS];
    // the tile's scanned totals of this lane's rows, asked for now and used after the chunk sums (volatile: not sunk to the use)
    double tq = 0.0, tp = 0.0;
    if (c < NS) {
        asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(tq) : "l"(tot + (size_t)(RB + c) * tiles + tile));
        asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(tp) : "l"(tot + (size_t)(RB + NS + c) * tiles + tile));
    }
    // M5a: chunk sums (recomputed, never stored in HBM), then the exclusive scans along the 32 chunks of the tile in shared
    // memory, lane = row, serial in chunk order (q rows inside-out, p rows outside-in; the loads do not depend on the
    // running sum, so the chain is 32 DADDs).  The p prefixes wait in V while the forward walk runs.
    {
        double pq[NS];
        mex_chunk_sums<LMAX, G, false>(rec_tile, c, s, pq);
#pragma unroll
        for (int i = 0; i < NS; ++i) V[i * kVStride + c] = s[i];
        __syncwarp();
        if (c < NS) {
            double* v = V + c * kVStride;
            double x[kMexThreads];
#pragma unroll
            for (int j = 0; j < kMexThreads; ++j) x[j] = v[j];
            double run = tq;   // the tile's exclusive prefix over the preceding tiles
#pragma unroll
            for (int j = 0; j < kMexThreads; ++j) { v[j] = run; run += x[j]; }
        }
        __syncwarp();
#pragma unroll
        for (int i = 0; i < NS; ++i) s[i] = V[i * kVStride + c];
        __syncwarp();
#pragma unroll
        for (int i = 0; i < NS; ++i) V[i * kVStride + c] = pq[i];
        __syncwarp();
        if (c < NS) {
            double* v = V + c * kVStride;
            double x[kMexThreads];
#pragma unroll
            for (int j = 0; j < kMexThreads; ++j) x[j] = v[j];
            double run = tp;
#pragma unroll
            for (int j = kMexThreads - 1; j >= 0; --j) { v[j] = run; run += x[j]; }
        }
        __syncwarp();
    }
    // inside-out: q
    {
        Rec p = load_rec(rec_tile, 0, c);
#pragma unroll(LMAX <= 6 ? 1 : 2)   // two particles in flight per walk pay at lmax >= 7 (N = 1e8, lmax 8: 18.0 -> 16.4 ms)
        for (int k = 0; k < kMexK; ++k) {
            const Rec nx = load_rec(rec_tile, (k + 1 < kMexK) ? k + 1 : k, c);
            double o[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) o[j] = sOut[(k * 4 + j) * kMexThreads + c];
            mex_eval_particle<LMAX, G, true, PO>(p, s, o);
#pragma unroll
            for (int j = 0; j < 4; ++j) sOut[(k * 4 + j) * kMexThreads + c] = o[j];
            p = nx;
        }
    }
    // outside-in: p
#pragma unroll
    for (int i = 0; i < NS; ++i) s[i] = V[i * kVStride + c];
    __syncwarp();   // V is free for the next group
    {
        Rec p = load_rec(rec_tile, kMexK - 1, c);
#pragma unroll(LMAX <= 6 ? 1 : 2)   // two particles in flight per walk pay at lmax >= 7 (N = 1e8, lmax 8: 18.0 -> 16.4 ms)
        for (int k = kMexK - 1; k >= 0; --k) {
            const Rec nx = load_rec(rec_tile, (k > 0) ? k - 1 : 0, c);
            double o[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) o[j] = sOut[(k * 4 + j) * kMexThreads + c];
            mex_eval_particle<LMAX, G, false, PO>(p, s, o);
#pragma unroll
            for (int j = 0; j < 4; ++j) sOut[(k * 4 + j) * kMexThreads + c] = o[j];
            p = nx;
        }
    }
}

__device__ __forceinline__ void st_global_v4(double* p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

#ifndef ETICS_EVAL_MINB
#define ETICS_EVAL_MINB 12
#endif
template <int LMAX, bool PO>
__global__ void __launch_bounds__(kMexThreads, LMAX <= 6 ? ETICS_EVAL_MINB : 8)
mex_evaluate_kernel(const double* __restrict__ rec, const unsigned* __restrict__ idxT, const double* __restrict__ tot,
                    long long tiles, long long N, double* __restrict__ out4) {
    __shared__ double sOut[kMexK * 4 * kMexThreads];
    __shared__ double V[mex_max_group_slots(LMAX) * kVStride];
    const long long tile = blockIdx.x;
    const int c = threadIdx.x;
    const double* rec_tile = rec + (size_t)tile * kRecFields * kMexTile;
    // the tile's records (7 fields x 256 doubles = 112 lines) are on their way before the first chunk sum asks for them
    // (N = 1e6: 120.2 -> 116.2 us)
#pragma unroll
    for (int i = c; i < 7 * kMexTile / 16; i += kMexThreads)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(rec_tile + 16 * i));
#pragma unroll
    for (int i = 0; i < kMexK * 4; ++i) sOut[i * kMexThreads + c] = 0.0;   // lane-private column: no barrier needed
    constexpr int NG = mex_num_groups(LMAX);
    mex_evaluate_group<LMAX, 0, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 1) mex_evaluate_group<LMAX, 1, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 2) mex_evaluate_group<LMAX, 2, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 3) mex_evaluate_group<LMAX, 3, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 4) mex_evaluate_group<LMAX, 4, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 5) mex_evaluate_group<LMAX, 5, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 6) mex_evaluate_group<LMAX, 6, PO>(rec_tile, sOut, V, tot, tiles, tile);
    if constexpr (NG > 7) mex_evaluate_group<LMAX, 7, PO>(rec_tile, sOut, V, tot, tiles, tile);
    // M7: transform and scatter.  All indices and the four angle fields of the chunk's records are loaded first (the sums are
    // dead, the registers are free): with one particle at a time every iteration waited out a full L2 round trip (ncu: 17 % of the
    // kernel's stall samples sat on this loop's first arithmetic).
    unsigned idx[kMexK];
    double gct[kMexK], gst[kMexK], gcp[kMexK], gsp[kMexK];
#pragma unroll
    for (int k = 0; k < kMexK; ++k) {
        idx[k] = idxT[(size_t)tile * kMexTile + k * kMexThreads + c];
        if (!PO) {
            const double* b = rec_tile + k * kMexThreads + c;
            gct[k] = b[2 * kMexTile]; gst[k] = b[3 * kMexTile]; gcp[k] = b[4 * kMexTile]; gsp[k] = b[5 * kMexTile];
        }
    }
#pragma unroll
    for (int k = 0; k < kMexK; ++k) {
        const long long p = tile * kMexTile + (long long)c * kMexK + k;
        if (p >= N) continue;
        if (PO) {   // out4 is the caller's pot array: one 8-byte store at the original index
            out4[idx[k]] = sOut[(k * 4 + 0) * kMexThreads + c];
            continue;
        }
        Geom g;
        g.r = 0.0; g.rinv = 0.0; g.ct = gct[k]; g.st = gst[k]; g.cp = gcp[k]; g.sp = gsp[k];
        double ax, ay, az;
        to_cartesian(g, sOut[(k * 4 + 1) * kMexThreads + c], sOut[(k * 4 + 2) * kMexThreads + c],
                     sOut[(k * 4 + 3) * kMexThreads + c], ax, ay, az);
        // ONE full 32-byte sector per particle at its original index (four 8-byte stores into the SoA outputs cost
        // 22 us of the kernel's 120 at N = 10^6 and 5 of 22 ms at N = 10^8); mex_unpack_kernel streams it into acc, pot
        st_global_v4(out4 + 4 * (size_t)idx[k], sOut[(k * 4 + 0) * kMexThreads + c], ax, ay, az);
    }
}

// (Phi, ax, ay, az) records by original index -> pot (N), acc (3,N).  Streaming: 32 B read + 32 B written per particle.
static __global__ void __launch_bounds__(256)
mex_unpack_kernel(const double2* __restrict__ out4, long long N, double* __restrict__ acc, double* __restrict__ pot) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double2 a = out4[2 * i], b = out4[2 * i + 1];
    if (pot) pot[i] = a.x;   // null: force only
    acc[i] = a.y;
    acc[N + i] = b.x;
    acc[2 * N + i] = b.y;
}

// ---------------------------------------------------------------------------------------------------------
// Host side.
// ---------------------------------------------------------------------------------------------------------
#if ETICS_MEX_PART == 0
cudaError_t mex_sort_launch(const double* pos, long long N, unsigned long long* keys_sorted, unsigned int* perm,
                            void* ws, cudaStream_t st) {
    const MexLayout L = make_mex_layout(N, 0);
    return mex_sort_enqueue(pos, nullptr, N, L, static_cast<char*>(ws), perm, keys_sorted, false, st, nullptr);
}

#endif   // ETICS_MEX_PART == 0

static RowDirs mex_row_dirs(int lmax) {
    RowDirs rd{};
    rd.ng = mex_num_groups(lmax);
    for (int g = 0; g < rd.ng; ++g) { rd.rb[g] = mex_row_base(lmax, g); rd.ns[g] = mex_group_slots(lmax, g); }
    return rd;
}

// phase 0: the whole sequence (etics_mex_force).  Radius-partitioned MEX splits it at the one point where the shards
// exchange: phase 1 = gather + tile totals + the shard's moment vector (totals), phase 2 = tile scan starting from `base`,
// evaluation, unpack.
template <int LMAX>
static cudaError_t mex_scan_enqueue(const MexLayout& L, char* ws, long long N, int what, double* acc, double* pot, cudaStream_t st,
                                    cudaEvent_t* ev, int phase, const double* base, double* totals) {
    double* rec = reinterpret_cast<double*>(ws + L.off_rec);
    unsigned* idxT = reinterpret_cast<unsigned*>(ws + L.off_idxT);
    double* tot = reinterpret_cast<double*>(ws + L.off_tot);
    cudaError_t e = cudaSuccess;
    if (phase != 2) {
        mex_gather_totals_kernel<LMAX><<<(unsigned)L.tiles, kMexThreads, 0, st>>>(
            reinterpret_cast<const double2*>(ws + L.off_pk), reinterpret_cast<const unsigned*>(ws + L.off_perm), N, L.tiles, rec, idxT, tot);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        if (ev) { cudaEventRecord(ev[3], st); cudaEventRecord(ev[4], st); }
    }
    if (phase == 1) {
        mex_rowtotal_kernel<<<mex_total_rows(LMAX), kTileScanThreads, 0, st>>>(tot, L.tiles, totals);
        return cudaGetLastError();
    }
    mex_tilescan_kernel<<<mex_total_rows(LMAX), kTileScanThreads, 0, st>>>(tot, L.tiles, mex_row_dirs(LMAX), base);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (ev) cudaEventRecord(ev[5], st);
    if (what == ETICS_WHAT_POTENTIAL) {
        mex_evaluate_kernel<LMAX, true><<<(unsigned)L.tiles, kMexThreads, 0, st>>>(rec, idxT, tot, L.tiles, N, pot);
        e = cudaGetLastError();
    } else {
        double* out4 = reinterpret_cast<double*>(ws + L.off_pk);   // the packed inputs were consumed by the gather
        mex_evaluate_kernel<LMAX, false><<<(unsigned)L.tiles, kMexThreads, 0, st>>>(rec, idxT, tot, L.tiles, N, out4);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        mex_unpack_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(reinterpret_cast<const double2*>(out4), N, acc,
                                                                          what == ETICS_WHAT_FORCE ? nullptr : pot);
        e = cudaGetLastError();
    }
    if (ev) cudaEventRecord(ev[6], st);
    return e;
}

// The scan launch sequence of one lmax range per translation unit.
#define ETICS_SCAN_ARGS const MexLayout &L, char *ws, long long N, int lmax, int what, double *acc, double *pot, cudaStream_t st, cudaEvent_t *ev, \
                        int phase, const double *base, double *totals
cudaError_t mex_scan_part0(ETICS_SCAN_ARGS);
cudaError_t mex_scan_part1(ETICS_SCAN_ARGS);
cudaError_t mex_scan_part2(ETICS_SCAN_ARGS);
cudaError_t mex_scan_part3(ETICS_SCAN_ARGS);
#define ETICS_CASE(LM) case LM: return mex_scan_enqueue<LM>(L, ws, N, what, acc, pot, st, ev, phase, base, totals);
#if ETICS_MEX_PART == 0
cudaError_t mex_scan_part0(ETICS_SCAN_ARGS) {
    switch (lmax) {
        ETICS_CASE(0) ETICS_CASE(1) ETICS_CASE(2) ETICS_CASE(3) ETICS_CASE(4) ETICS_CASE(5) ETICS_CASE(6)
        default: return cudaErrorInvalidValue;
    }
}
#elif ETICS_MEX_PART == 1
cudaError_t mex_scan_part1(ETICS_SCAN_ARGS) {
    switch (lmax) {
        ETICS_CASE(7) ETICS_CASE(8)
        default: return cudaErrorInvalidValue;
    }
}
#elif ETICS_MEX_PART == 2
cudaError_t mex_scan_part2(ETICS_SCAN_ARGS) {
    switch (lmax) {
        ETICS_CASE(9)
        default: return cudaErrorInvalidValue;
    }
}
#else
cudaError_t mex_scan_part3(ETICS_SCAN_ARGS) {
    switch (lmax) {
        ETICS_CASE(10)
        default: return cudaErrorInvalidValue;
    }
}
#endif
#undef ETICS_CASE

#if ETICS_MEX_PART == 0
// ev (optional): 7 events recorded at: start, after keygen, after the radix passes, after gather, after aggregate,
// after tilescan, after evaluate.
static cudaError_t mex_scan_dispatch(ETICS_SCAN_ARGS) {
    if (lmax <= 6) return mex_scan_part0(L, ws, N, lmax, what, acc, pot, st, ev, phase, base, totals);
    if (lmax <= 8) return mex_scan_part1(L, ws, N, lmax, what, acc, pot, st, ev, phase, base, totals);
    if (lmax == 9) return mex_scan_part2(L, ws, N, lmax, what, acc, pot, st, ev, phase, base, totals);
    return mex_scan_part3(L, ws, N, lmax, what, acc, pot, st, ev, phase, base, totals);
}

static cudaError_t mex_force_enqueue(const double* pos, const double* mass, long long N, int lmax, int what,
                                     double* acc, double* pot, void* wsv, cudaStream_t st, cudaEvent_t* ev) {
    const MexLayout L = make_mex_layout(N, lmax);
    char* ws = static_cast<char*>(wsv);
    unsigned* idxA = reinterpret_cast<unsigned*>(ws + L.off_perm);
    if (ev) cudaEventRecord(ev[0], st);
    cudaError_t e = mex_sort_enqueue(pos, mass, N, L, ws, idxA, nullptr, true, st, ev ? ev[1] : nullptr);
    if (e != cudaSuccess) return e;
    if (ev) cudaEventRecord(ev[2], st);
    return mex_scan_dispatch(L, ws, N, lmax, what, acc, pot, st, ev, 0, nullptr, nullptr);
}

// ---- radius-partitioned MEX: the sequence above cut at the exchange of the shards' moment vectors -----------------------
int mex_shard_rows(int lmax) { return mex_total_rows(lmax); }

cudaError_t mex_shard_moments_launch(const double* pos, const double* mass, long long N, int lmax, double* totals, void* wsv,
                                     cudaStream_t st) {
    const MexLayout L = make_mex_layout(N, lmax);
    char* ws = static_cast<char*>(wsv);
    cudaError_t e = mex_sort_enqueue(pos, mass, N, L, ws, reinterpret_cast<unsigned*>(ws + L.off_perm), nullptr, true, st, nullptr);
    if (e != cudaSuccess) return e;
    return mex_scan_dispatch(L, ws, N, lmax, ETICS_WHAT_BOTH, nullptr, nullptr, st, nullptr, 1, nullptr, totals);
}

cudaError_t mex_shard_bases_launch(const double* parts, int nparts, int rank, int lmax, double* base, cudaStream_t st) {
    const int rows = mex_total_rows(lmax);
    mex_shard_bases_kernel<<<(rows + 127) / 128, 128, 0, st>>>(parts, nparts, rank, rows, mex_row_dirs(lmax), base);
    return cudaGetLastError();
}

cudaError_t mex_shard_force_launch(long long N, int lmax, int what, const double* base, double* acc, double* pot, void* wsv,
                                   cudaStream_t st) {
    const MexLayout L = make_mex_layout(N, lmax);
    return mex_scan_dispatch(L, static_cast<char*>(wsv), N, lmax, what, acc, pot, st, nullptr, 2, base, nullptr);
}

cudaError_t mex_force_launch(const double* pos, const double* mass, long long N, int lmax, int what,
                             double* acc, double* pot, void* ws, cudaStream_t st) {
    return mex_force_enqueue(pos, mass, N, lmax, what, acc, pot, ws, st, nullptr);
}

// Measurement support: the same launch sequence with CUDA events between the stages; synchronises the stream.
cudaError_t mex_force_timed(const double* pos, const double* mass, long long N, int lmax, double* acc, double* pot,
                            void* ws, cudaStream_t st, float* stage_ms) {
    cudaEvent_t ev[7] = {};
    cudaError_t e = cudaSuccess;
    for (auto& x : ev) { e = cudaEventCreate(&x); if (e != cudaSuccess) break; }
    if (e == cudaSuccess) e = mex_force_enqueue(pos, mass, N, lmax, ETICS_WHAT_BOTH, acc, pot, ws, st, ev);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess)
        for (int i = 0; i < 6; ++i) cudaEventElapsedTime(&stage_ms[i], ev[i], ev[i + 1]);
    for (auto& x : ev) if (x) cudaEventDestroy(x);
    return e;
}

#endif   // ETICS_MEX_PART == 0

}  // namespace etics

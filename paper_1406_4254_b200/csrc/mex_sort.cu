// mex_sort.cu — MEX steps M1–M2: radial sort of the particles by r^2 (§3.2: "the
// distance square ... for the sorting operation"), stable, ties broken by particle index.  Hand-written for
// sm_100a, no CUB/Thrust.
//
// The paper sorts whole particle structs with Thrust's merge sort.  Here the sort moves ONE 64-bit
// word per particle, word_k = (prefix_k << ibits) | k with prefix_k = (key_k - kmin) >> shift: the leading B bits of the
// key's offset from the smallest key above the ibits = bits(N-1) bits of the particle index.  The words go through
// stable LSD passes over digits of the prefix (the index bits ride along); particles whose prefixes collide (the
// key bits below `shift` were not sorted) form short runs that a fix-up orders by (full key, index).
//
// Every pass is histogram -> scan -> scatter over SEGMENTS (consecutive tiles owned by one block): no block ever
// waits for another block's progress, and everything is integer work in a fixed order.
//   N <= one tile per resident block (~1.2e6): ONE cooperative kernel, grid-wide barriers between the phases, B = 33,
//     three 11-bit passes (the sort is a single wave and latency-bound: fewer, wider passes).
//   larger N: one kernel per phase, B = 36, four 9-bit passes over 5120-word tiles, two scatter blocks per SM (bandwidth-bound:
//     with 2048 digit values a tile scatters runs of two words; 512 values give 80-byte runs).
//   mex_sort_fallback_kernel: a run longer than kFixMaxRun (many particles within 2^shift ulps of each other, yet not
//     all equal: e.g. two thin shells) raises a flag and this plain single-block LSD sort of the full keys redoes the
//     job — correct for any input, slow, never taken by the paper's workloads.
#include <cooperative_groups.h>

#include <cstdlib>

#include "mex_common.cuh"

namespace cg = cooperative_groups;

namespace etics {

// =========================================================================================================
// Sort plan: a pure function of (kmin, kmax, N), recomputed by every kernel from the header.
// =========================================================================================================
struct SortPlan {
    unsigned long long kmin;
    int ibits;      // bits of the particle index inside a word
    int shift;      // key bits below the prefix
    int B;          // prefix bits
    int passes;     // 0..kSortMaxPasses
    // digit of pass i: word bits [ibits + lo(i), ibits + lo(i) + w(i)); the B bits are spread evenly over the passes
    __host__ __device__ int w(int i) const { return i < passes ? B / passes + (i < B % passes ? 1 : 0) : 0; }
    __host__ __device__ int lo(int i) const { return i < passes ? i * (B / passes) + (i < B % passes ? i : B % passes) : B; }
};

__host__ __device__ inline int bit_length64(unsigned long long v) {
    int n = 0;
    while (v) { ++n; v >>= 1; }
    return n;
}

__host__ __device__ inline SortPlan make_sort_plan(unsigned long long kmin, unsigned long long kmax, long long N,
                                                   int prefix_bits, int digit_bits) {
    SortPlan p;
    p.kmin = kmin;
    p.ibits = bit_length64((unsigned long long)(N - 1));
    const int nbits = bit_length64(kmax - kmin);
    p.B = nbits < prefix_bits ? nbits : prefix_bits;
    p.shift = nbits - p.B;
    p.passes = (p.B + digit_bits - 1) / digit_bits;
    return p;
}

__device__ __forceinline__ SortPlan load_plan(const SortHeader* hdr, long long N, int prefix_bits, int digit_bits) {
    const unsigned long long inv = __ldcg(&hdr->inv_kmin), kmax = __ldcg(&hdr->kmax);
    return make_sort_plan(~inv, kmax, N, prefix_bits, digit_bits);
}

// =========================================================================================================
// M1: keys, packed particle records, min/max key.
// =========================================================================================================
__device__ __forceinline__ unsigned long long mex_key(double x, double y, double z) {
    double t = __dmul_rn(x, x);
    t = __fma_rn(y, y, t);
    t = __fma_rn(z, z, t);
    return (unsigned long long)__double_as_longlong(t);   // r^2 >= 0: the bit pattern is monotone in r^2
}

// =========================================================================================================
// M1–M2 in ONE persistent cooperative kernel (grid = every block the GPU holds at once; grid-wide barriers
// between the phases, no polling on other blocks' progress anywhere):
//
//   phase K   keys, (x,y,z,m) records, min / max key (integer atomics)
//   phase W   packed words; digit histogram of pass 0 per SEGMENT (a segment = the consecutive tiles one block owns)
//   per pass: phase S   exclusive scan of the segment histograms along the segments, one warp per digit value
//             phase P   every block walks its tiles in order: rank inside the tile (stable), positions from the
//                       segment's scanned offsets plus a running count per digit, one coalesced write
//             phase H   segment histograms of the next pass's digit
//   phase F   fix-up of colliding prefixes -> permutation (and sorted keys)
//
// Everything is integer work in a fixed order, so the result is unique.  Data written by one block and read by
// another after a barrier is read with ld.global.cg (L2), never through the non-coherent path.
// =========================================================================================================
struct SortParams {
    const double* pos;
    const double* mass;
    long long N;
    unsigned long long* keys;
    double2* pk;              // null: no records
    SortHeader* hdr;
    unsigned long long* bufA;
    unsigned long long* bufB;
    unsigned* seg_hist;       // [nseg][kSortBins]
    unsigned* bin_tot;        // [kSortBins]
    unsigned* perm;
    unsigned* itmp;           // second index buffer of the fallback sort
    unsigned long long* keys_sorted;   // may be null
    long long tiles, tps;     // tiles (kSortTile words in the single-wave sort, kSortThreads * kLargeItems above); tiles per segment
    int nseg;
    int prefix_bits, digit_bits;   // key bits that are radix-sorted; width of a digit (<= kSortDigitBits)
};

constexpr int kSortItems = 16;                             // single-wave sort: 4096-word tiles
constexpr int kSortTile = kSortThreads * kSortItems;
static_assert(kSortTile == kSortMinTile, "workspace sizing");
// Bandwidth-bound sort: words per thread and tile.  N = 1e8, whole sort: 16 words with 3 blocks per SM (80 registers) 5.07 ms;
// with 2 blocks per SM (128 registers, no spills): 16 -> 4.84, 20 -> 4.745, 22 -> 4.74, 24 -> 4.77, 28 -> 4.73 (spills), 32 with
// one block per SM 5.32.  Fewer resident blocks mean fewer open write frontiers (segments x 512 digit values) in L2 and
// longer runs of equal digits per tile (20 words x 256 threads / 512 values = 80 bytes).
constexpr int kLargeItems = 20;
constexpr int kLargeMinBlocks = 2;
static_assert(kLargeItems >= kSortItems && kLargeItems * kSortThreads < 65536, "workspace sizing; 16-bit tile positions");
constexpr int kScanStrip = 8;                              // digit values per strip of the segment scan (one 32-byte sector)

// DB = bits of a digit (compile time: 11 for the single-wave sort, 9 for the bandwidth-bound one).
template <int DB, int ITEMS = kSortItems>
struct SortSmem {
    static constexpr int BINS = 1 << DB;
    static constexpr int BPT = BINS / kSortThreads;   // thread t owns digits BPT t .. BPT t + BPT - 1 in the offset steps
    static_assert(BPT >= 2 && BPT % 2 == 0 && DB <= kSortDigitBits, "16-bit counters are moved in 32-bit pairs");
    unsigned short cnt[kSortWarps][BINS];   // ranking: [tag | count]; afterwards position of (warp, digit) inside the tile
    unsigned gbase[BINS];                   // global position of the tile's first word of digit d, minus its tile position
    unsigned run[BINS];                     // scatter: next free global position of digit d for this segment; histogram phases: counts
    unsigned scan_tmp[kSortWarps];
    unsigned long long red[2][kSortWarps];
    unsigned long long stage[kSortThreads * ITEMS];    // scatter: the tile in output order; scan: a strip of the segment histograms
};

template <int W>
__device__ __forceinline__ void ld_words(const unsigned* p, unsigned (&v)[W]) {
    if constexpr (W % 4 == 0) {
#pragma unroll
        for (int i = 0; i < W / 4; ++i) {
            const uint4 t = reinterpret_cast<const uint4*>(p)[i];
            v[4 * i] = t.x; v[4 * i + 1] = t.y; v[4 * i + 2] = t.z; v[4 * i + 3] = t.w;
        }
    } else if constexpr (W % 2 == 0) {
#pragma unroll
        for (int i = 0; i < W / 2; ++i) {
            const uint2 t = reinterpret_cast<const uint2*>(p)[i];
            v[2 * i] = t.x; v[2 * i + 1] = t.y;
        }
    } else {
#pragma unroll
        for (int i = 0; i < W; ++i) v[i] = p[i];
    }
}
template <int W>
__device__ __forceinline__ void st_words(unsigned* p, const unsigned (&v)[W]) {
    if constexpr (W % 4 == 0) {
#pragma unroll
        for (int i = 0; i < W / 4; ++i) reinterpret_cast<uint4*>(p)[i] = make_uint4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
    } else if constexpr (W % 2 == 0) {
#pragma unroll
        for (int i = 0; i < W / 2; ++i) reinterpret_cast<uint2*>(p)[i] = make_uint2(v[2 * i], v[2 * i + 1]);
    } else {
#pragma unroll
        for (int i = 0; i < W; ++i) p[i] = v[i];
    }
}
template <int W>
__device__ __forceinline__ void ldcg_words(const unsigned* p, unsigned (&v)[W]) {
    if constexpr (W % 4 == 0) {
#pragma unroll
        for (int i = 0; i < W / 4; ++i) {
            const uint4 t = __ldcg(reinterpret_cast<const uint4*>(p) + i);
            v[4 * i] = t.x; v[4 * i + 1] = t.y; v[4 * i + 2] = t.z; v[4 * i + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int i = 0; i < W / 2; ++i) {
            const uint2 t = __ldcg(reinterpret_cast<const uint2*>(p) + i);
            v[2 * i] = t.x; v[2 * i + 1] = t.y;
        }
    }
}

template <bool SYNC_AFTER = true>
__device__ __forceinline__ unsigned block_exclusive_scan_256(unsigned v, unsigned* tmp) {
    // kSortThreads == 256 threads, one value each
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) tmp[warp] = inc;
    __syncthreads();
    unsigned woff = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) {
        const unsigned t = tmp[w];
        if (w < warp) woff += t;
    }
    if constexpr (SYNC_AFTER) __syncthreads();   // tmp may be rewritten by a caller that does not pass another barrier first
    return woff + inc - v;
}

constexpr int kKeygenItems = 4;

// phase K
__device__ __forceinline__ void sort_phase_keys(const SortParams& P, unsigned long long (*red)[kSortWarps]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long N = P.N;
    unsigned long long inv = 0, mx = 0;
    const long long stride = (long long)gridDim.x * kSortThreads * kKeygenItems;
    for (long long base = (long long)blockIdx.x * kSortThreads * kKeygenItems; base < N; base += stride) {
        double x[kKeygenItems], y[kKeygenItems], z[kKeygenItems], mk[kKeygenItems];
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * kSortThreads + threadIdx.x;
            const bool ok = k < N;
            x[j] = ok ? P.pos[k] : 0.0; y[j] = ok ? P.pos[N + k] : 0.0; z[j] = ok ? P.pos[2 * N + k] : 0.0;
            mk[j] = (ok && P.pk) ? P.mass[k] : 0.0;
        }
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * kSortThreads + threadIdx.x;
            if (k < N) {
                const unsigned long long key = mex_key(x[j], y[j], z[j]);
                P.keys[k] = key;
                inv = max(inv, ~key);
                mx = max(mx, key);
            }
            // The warp's 32 records are 1024 contiguous bytes: two fully coalesced 16-byte stores per lane (lane l writes the
            // (x,y) or (z,m) half of the record of lane l / 2, then of lane 16 + l / 2) instead of two stores that each touch
            // half of 32 sectors (N = 1e8: 4.86 -> 4.77 ms).
            if (P.pk) {
                const long long k0 = base + j * kSortThreads + (threadIdx.x & ~31);   // the warp's first particle
                const bool hi = lane & 1;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int src = 16 * h + (lane >> 1);
                    const double ax = __shfl_sync(0xffffffffu, x[j], src), ay = __shfl_sync(0xffffffffu, y[j], src);
                    const double az = __shfl_sync(0xffffffffu, z[j], src), am = __shfl_sync(0xffffffffu, mk[j], src);
                    if (k0 + src < N) P.pk[2 * (k0 + src) + (hi ? 1 : 0)] = hi ? make_double2(az, am) : make_double2(ax, ay);
                }
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        inv = max(inv, __shfl_xor_sync(0xffffffffu, inv, o));
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if (lane == 0) { red[0][warp] = inv; red[1][warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < kSortWarps; ++w) { inv = max(inv, red[0][w]); mx = max(mx, red[1][w]); }
        atomicMax(&P.hdr->inv_kmin, inv);   // integer atomics: the result does not depend on their order
        atomicMax(&P.hdr->kmax, mx);
    }
}

// phases W (FIRST: words are built from the keys and stored) and H: digit histogram of this block's segment
// TILE: words per tile (a compile-time constant in both kernels that call this)
template <bool FIRST, int TILE>
__device__ __forceinline__ void sort_phase_hist(const SortParams& P, unsigned* hist, int bins, const SortPlan& pl, int pass,
                                                const unsigned long long* in) {
    const int seg = blockIdx.x;
    if (seg >= P.nseg) return;
    const int dshift = pl.ibits + pl.lo(pass);
    const unsigned dmask = (1u << pl.w(pass)) - 1u;
    for (int i = threadIdx.x; i < bins; i += kSortThreads) hist[i] = 0u;
    __syncthreads();
    const long long k0 = (long long)seg * P.tps * TILE;
    long long k1 = k0 + P.tps * TILE;
    if (k1 > P.N) k1 = P.N;
    for (long long base = k0; base < k1; base += kSortThreads * kKeygenItems) {
        unsigned long long w[kKeygenItems];
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * kSortThreads + threadIdx.x;
            w[j] = (k < k1) ? __ldcg((FIRST ? P.keys : in) + k) : 0ull;
        }
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * kSortThreads + threadIdx.x;
            if (k < k1) {
                if (FIRST) {
                    w[j] = (((w[j] - pl.kmin) >> pl.shift) << pl.ibits) | (unsigned long long)k;
                    P.bufA[k] = w[j];
                }
                if (pass < pl.passes) atomicAdd(&hist[(unsigned)(w[j] >> dshift) & dmask], 1u);
            }
        }
    }
    __syncthreads();
    unsigned* row = P.seg_hist + (size_t)seg * kSortBins;
    for (int i = threadIdx.x; i < bins; i += kSortThreads) row[i] = hist[i];
}

// phase S: seg_hist[seg][d] -> exclusive prefix over the segments; bin_tot[d] = total.  Block b owns the strip of
// kScanStrip = 8 digit values 8b..8b+7 (one 32-byte sector per segment row): the strip is loaded in one round
// trip, warp w scans column w in shared memory, the strip is stored back.
__device__ __forceinline__ void sort_phase_scan(const SortParams& P, unsigned* strip /* [nseg][8] */, int bins) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    static_assert(kScanStrip == kSortWarps, "warp w scans column w of the strip");
    for (int b = blockIdx.x; b < bins / kScanStrip; b += gridDim.x) {
        for (int s = tid; s < P.nseg; s += kSortThreads) {
            const uint4* row = reinterpret_cast<const uint4*>(P.seg_hist + (size_t)s * kSortBins + kScanStrip * b);
            const uint4 v0 = __ldcg(row), v1 = __ldcg(row + 1);
            reinterpret_cast<uint4*>(strip + 8 * s)[0] = v0;
            reinterpret_cast<uint4*>(strip + 8 * s)[1] = v1;
        }
        __syncthreads();
        {
            unsigned carry = 0;
            for (int s0 = 0; s0 < P.nseg; s0 += 32) {
                const int s = s0 + lane;
                const unsigned v = (s < P.nseg) ? strip[8 * s + warp] : 0u;
                unsigned inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                if (s < P.nseg) strip[8 * s + warp] = carry + inc - v;
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) P.bin_tot[kScanStrip * b + warp] = carry;
        }
        __syncthreads();
        for (int s = tid; s < P.nseg; s += kSortThreads) {
            uint4* row = reinterpret_cast<uint4*>(P.seg_hist + (size_t)s * kSortBins + kScanStrip * b);
            row[0] = reinterpret_cast<const uint4*>(strip + 8 * s)[0];
            row[1] = reinterpret_cast<const uint4*>(strip + 8 * s)[1];
        }
        __syncthreads();
    }
}

// phase P: stable scatter of this block's segment by the digit of `pass`.
// Tile = 256 threads x 16 words, loaded warp-striped (item i of warp w at tile base + w*512 + 32 i + lane), so the
// order (warp, item, lane) is the order of the input.
// Ranking: per warp and digit a 16-bit counter [tag:5 | count:11].  For every item the lanes stamp their lane
// number on their digit's counter and read it back: if every lane finds its own stamp, all 32 digits of the item
// are distinct (78 % of the items for uniformly distributed 11-bit digits) and the rank is simply the counter;
// otherwise the lanes that share a digit find each other with one ballot per digit bit.  (Measured in round 1:
// MATCH.ANY iterates over the distinct values of a warp, ~230 cycles for random digits; shared-memory atomics do
// not return ranks in lane order.)
template <int DB, int ITEMS>
__device__ __forceinline__ void sort_phase_scatter(const SortParams& P, SortSmem<DB, ITEMS>& S, const SortPlan& pl, int pass,
                                                   const unsigned long long* in, unsigned long long* out) {
    constexpr int BINS = SortSmem<DB, ITEMS>::BINS, BPT = SortSmem<DB, ITEMS>::BPT, WPT = BPT / 2;
    constexpr int kSortItems = ITEMS, kSortTile = kSortThreads * ITEMS;   // (shadow the single-wave constants)
    const int seg = blockIdx.x;
    if (seg >= P.nseg) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long N = P.N;
    const int dshift = pl.ibits + pl.lo(pass);
    const unsigned dmask = (1u << pl.w(pass)) - 1u;

    // first global position of every digit for this segment: exclusive scan of the totals + the segment's offset
    {
        unsigned hb[BPT], of[BPT];
        ldcg_words<BPT>(P.bin_tot + BPT * tid, hb);
        ldcg_words<BPT>(P.seg_hist + (size_t)seg * kSortBins + BPT * tid, of);
        unsigned run = 0;
#pragma unroll
        for (int q = 0; q < BPT; ++q) { const unsigned t = hb[q]; hb[q] = run; run += t; }
        const unsigned off = block_exclusive_scan_256(run, S.scan_tmp);
#pragma unroll
        for (int q = 0; q < BPT; ++q) S.run[BPT * tid + q] = hb[q] + off + of[q];
    }

    const long long t0 = (long long)seg * P.tps;
    long long t1 = t0 + P.tps;
    if (t1 > P.tiles) t1 = P.tiles;
    const unsigned lt_mask = (1u << lane) - 1u;
    unsigned long long key[kSortItems];
    auto load_tile = [&](long long tile) {
        const long long base = tile * kSortTile + (long long)warp * (32 * kSortItems);
        const unsigned long long* src = in + base + lane;
        if ((tile + 1) * kSortTile <= N) {   // every tile but the last one: no bounds checks
#pragma unroll
            for (int i = 0; i < kSortItems; ++i) key[i] = __ldcg(src + 32 * i);
        } else {
#pragma unroll
            for (int i = 0; i < kSortItems; ++i) {
                const long long k = base + 32 * i + lane;
                key[i] = (k < N) ? __ldcg(in + k) : ~0ull;   // padding sorts last in every pass and is never written (position >= N)
            }
        }
    };
    // each warp clears its own counter row (1 << DB 16-bit counters): before the first tile, and again once the row has
    // been used for the last time in a tile (below) — no block barrier is needed for it
    auto clear_own_counters = [&]() {
        uint4* c = reinterpret_cast<uint4*>(&S.cnt[warp][0]);
        constexpr int kVec = BINS * 2 / 16;
        static_assert(kVec % 32 == 0, "counter clearing");
#pragma unroll
        for (int i = 0; i < kVec / 32; ++i) c[i * 32 + lane] = make_uint4(0u, 0u, 0u, 0u);
        __syncwarp();
    };
    clear_own_counters();
    load_tile(t0);
    for (long long tile = t0; tile < t1; ++tile) {
        // the tile after this one is loaded while this one is written: bring it into L2 now (one 128-byte line per thread)
        if (tile + 1 < t1) {
#pragma unroll
            for (int h = 0; h < (kSortItems + 15) / 16; ++h) {
                const int w = (h * kSortThreads + tid) * 16;   // one 128-byte line per thread and round
                const long long k = (tile + 1) * kSortTile + w;
                if ((kSortItems % 16 == 0 || w < kSortTile) && k < N) asm volatile("prefetch.global.L2 [%0];" :: "l"(in + k));
            }
        }

        // ---- rank ---------------------------------------------------------------------------------------------
        unsigned short rank[kSortItems];
        volatile unsigned short* cw = S.cnt[warp];
        if constexpr (DB > 9) {
            // wide digits: most items have 32 distinct digits — stamp, read back, and only on a collision find the peers
#pragma unroll
            for (int i = 0; i < kSortItems; ++i) {
                const unsigned d = (unsigned)(key[i] >> dshift) & dmask;
                const unsigned c = cw[d] & 0x7ffu;
                __syncwarp();
                cw[d] = (unsigned short)((lane << 11) | c);
                __syncwarp();
                const bool own = (cw[d] >> 11) == (unsigned)lane;
                if (__all_sync(0xffffffffu, own)) {
                    rank[i] = (unsigned short)c;
                    cw[d] = (unsigned short)(c + 1u);
                } else {
                    unsigned peers = 0xffffffffu;
#pragma unroll
                    for (int b = 0; b < DB; ++b) {
                        const bool bit = (d >> b) & 1u;
                        const unsigned vote = __ballot_sync(0xffffffffu, bit);
                        peers &= bit ? vote : ~vote;
                    }
                    const unsigned lower = peers & lt_mask;
                    rank[i] = (unsigned short)(c + __popc(lower));
                    if (lower == 0u) cw[d] = (unsigned short)(c + __popc(peers));
                }
                __syncwarp();
            }
        } else {
            // narrow digits: collisions are the rule — the lanes that share a digit find each other with one ballot per digit
            // bit; the lowest of them adds the group's size to the warp's counter of that digit (two 16-bit counters per
            // word: a 32-bit shared-memory atomic, the sums stay below 2^16) and hands the old count to the others.  The atomics
            // of successive items do not wait for one another's results; __syncwarp orders them (item by item: stable).
            unsigned* cw32 = reinterpret_cast<unsigned*>(&S.cnt[warp][0]);
#pragma unroll
            for (int i = 0; i < kSortItems; ++i) {
                const unsigned d = (unsigned)(key[i] >> dshift) & dmask;
                unsigned pe = 0xffffffffu;
#pragma unroll
                for (int b = 0; b < DB; ++b) {
                    const bool bit = (d >> b) & 1u;
                    const unsigned vote = __ballot_sync(0xffffffffu, bit);
                    pe &= bit ? vote : ~vote;
                }
                const unsigned lower = pe & lt_mask;
                const unsigned sh = (d & 1u) << 4;
                unsigned old = 0u;
                if (lower == 0u) old = atomicAdd(cw32 + (d >> 1), (unsigned)__popc(pe) << sh);
                __syncwarp();
                old = __shfl_sync(0xffffffffu, old, __ffs(pe) - 1);
                rank[i] = (unsigned short)(((old >> sh) & 0xffffu) + __popc(lower));
            }
        }
        __syncthreads();

        // ---- thread t owns BPT digits: per-warp counts -> exclusive over warps, tile totals -----------------------
        unsigned tot[BPT];
        {
            unsigned run[WPT];   // 16-bit running sums, two per word (<= kSortTile < 65536)
#pragma unroll
            for (int i = 0; i < WPT; ++i) run[i] = 0u;
#pragma unroll
            for (int w = 0; w < kSortWarps; ++w) {
                unsigned* p = reinterpret_cast<unsigned*>(&S.cnt[w][BPT * tid]);
                unsigned v[WPT];
                ld_words<WPT>(p, v);
                st_words<WPT>(p, run);
#pragma unroll
                for (int i = 0; i < WPT; ++i) run[i] += v[i] & 0x07ff07ffu;
            }
#pragma unroll
            for (int i = 0; i < WPT; ++i) { tot[2 * i] = run[i] & 0xffffu; tot[2 * i + 1] = run[i] >> 16; }
        }
        {
            unsigned loc[BPT];   // position of the tile's first word of digit d inside the tile
            unsigned run = 0;
#pragma unroll
            for (int q = 0; q < BPT; ++q) { loc[q] = run; run += tot[q]; }
            // no barrier after the scan: scan_tmp is not written again before the barriers of the next tile
            const unsigned off = block_exclusive_scan_256<false>(run, S.scan_tmp);
#pragma unroll
            for (int q = 0; q < BPT; ++q) loc[q] += off;
            unsigned add[WPT];
#pragma unroll
            for (int i = 0; i < WPT; ++i) add[i] = loc[2 * i] | (loc[2 * i + 1] << 16);
#pragma unroll
            for (int w = 0; w < kSortWarps; ++w) {
                unsigned* p = reinterpret_cast<unsigned*>(&S.cnt[w][BPT * tid]);
                unsigned v[WPT];
                ld_words<WPT>(p, v);
#pragma unroll
                for (int i = 0; i < WPT; ++i) v[i] += add[i];
                st_words<WPT>(p, v);
            }
#pragma unroll
            for (int q = 0; q < BPT; ++q) {
                const int d = BPT * tid + q;
                const unsigned r = S.run[d];
                S.gbase[d] = r - loc[q];
                S.run[d] = r + tot[q];
            }
        }
        __syncthreads();

        // ---- reorder inside the tile (stable), then write runs of equal digits ---------------------------------
#pragma unroll
        for (int i = 0; i < kSortItems; ++i) {
            const unsigned d = (unsigned)(key[i] >> dshift) & dmask;
            S.stage[S.cnt[warp][d] + rank[i]] = key[i];
        }
        if (tile + 1 < t1) load_tile(tile + 1);   // in flight while this tile is written
        __syncthreads();
        clear_own_counters();   // the row was last read by this warp's staging above
#pragma unroll
        for (int i = 0; i < kSortItems; ++i) {
            const unsigned j = i * kSortThreads + tid;
            const unsigned long long kk = S.stage[j];
            const unsigned d = (unsigned)(kk >> dshift) & dmask;
            const unsigned g = S.gbase[d] + j;
            if ((long long)g < N) out[g] = kk;
        }
        // no block barrier here: stage and gbase are rewritten only after the next tile's barriers, which every thread
        // reaches after this loop; the counters of the next ranking are this warp's own
    }
}

// phase F: order the runs of equal prefixes by (full key, index); write the permutation (and the sorted keys).
// Particles whose prefixes collide (the key bits below `shift` were not sorted) form short runs; the thread at the
// head of a run orders it.  A run longer than kFixMaxRun raises the fallback flag.
constexpr int kFixMaxRun = 32;

constexpr int kFixItems = 8;   // positions per thread and step: the loads of a step are issued together

__device__ __noinline__ void sort_fix_run(const SortParams& P, const SortPlan& pl, const unsigned long long* words,
                                          long long p, unsigned long long w) {
    const long long N = P.N;
    const unsigned long long imask = (1ull << pl.ibits) - 1ull;
    const unsigned long long pre = w >> pl.ibits;
    unsigned idx[kFixMaxRun];
    unsigned long long key[kFixMaxRun];
    int len = 0;
    while (p + len < N && len < kFixMaxRun) {
        const unsigned long long v = (len == 0) ? w : __ldcg(words + p + len);
        if ((v >> pl.ibits) != pre) break;
        idx[len] = (unsigned)(v & imask);
        ++len;
    }
    if (len == kFixMaxRun && p + len < N && (__ldcg(words + p + len) >> pl.ibits) == pre) {
        atomicExch(&P.hdr->fallback, 1u);   // too long to order here: the fallback sort redoes the whole job
        return;
    }
    for (int j = 0; j < len; ++j) key[j] = __ldcg(P.keys + idx[j]);
    // stable insertion sort by the full key: members arrive in index order (the passes are stable)
    for (int j = 1; j < len; ++j) {
        const unsigned long long kj = key[j];
        const unsigned ij = idx[j];
        int q = j - 1;
        while (q >= 0 && key[q] > kj) { key[q + 1] = key[q]; idx[q + 1] = idx[q]; --q; }
        key[q + 1] = kj; idx[q + 1] = ij;
    }
    for (int j = 0; j < len; ++j) {
        P.perm[p + j] = idx[j];
        if (P.keys_sorted) P.keys_sorted[p + j] = key[j];
    }
}

// phase F1: particles alone in their prefix are final; the heads of runs are listed (in the words buffer the last pass
// left free: any order, every head writes a range of its own) for phase F2.
__device__ __forceinline__ void sort_phase_fixup(const SortParams& P, const SortPlan& pl, const unsigned long long* words,
                                                 unsigned* heads) {
    // A warp takes kFixItems x 32 consecutive positions per step (item j, lane l: position p0 + 32 j + l).  "Position p and
    // p + 1 share a prefix" is one comparison per position; everything else — run to the left, alone, head of a run —
    // follows from the ballots of that bit, in warp-uniform registers.
    const long long N = P.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned long long lim = 1ull << pl.ibits;   // same prefix <=> (a ^ b) < lim;  ibits <= 31
    const unsigned imask = (unsigned)(lim - 1ull);
    const bool runs = pl.shift > 0;                     // all key bits sorted: no runs at all
    const unsigned lt_mask = (1u << lane) - 1u;
    constexpr long long kChunk = 32 * kFixItems;
    const long long stride = (long long)gridDim.x * kSortWarps * kChunk;
    for (long long p0 = ((long long)blockIdx.x * kSortWarps + warp) * kChunk; p0 < N; p0 += stride) {
        unsigned long long w[kFixItems];
#pragma unroll
        for (int j = 0; j < kFixItems; ++j) {
            const long long p = p0 + 32 * j + lane;
            w[j] = (p < N) ? __ldcg(words + p) : 0ull;
        }
        const unsigned long long el = (p0 > 0) ? __ldcg(words + p0 - 1) : 0ull;             // warp-uniform addresses
        const unsigned long long er = (p0 + kChunk < N) ? __ldcg(words + p0 + kChunk) : 0ull;
        // R[j]: bit l = the position of (item j, lane l) and the next position share a prefix.  Run to the left, head of a run
        // and alone follow from R (and c0: the same bit for the position before the chunk) in warp-uniform registers.
        unsigned R[kFixItems];
        const unsigned c0 = (runs && p0 > 0 && (((el ^ __shfl_sync(0xffffffffu, w[0], 0)) < lim))) ? 1u : 0u;
#pragma unroll
        for (int j = 0; j < kFixItems; ++j) {
            const long long p = p0 + 32 * j + lane;
            // lane l reads the word of lane l + 1; lane 31 reads lane 0's NEXT item (or the word after the chunk)
            const unsigned long long next0 = (j + 1 < kFixItems) ? w[(j + 1) % kFixItems] : er;
            const unsigned long long give = (lane == 0) ? next0 : w[j];
            const unsigned long long nb = __shfl_sync(0xffffffffu, give, (lane + 1) & 31);
            R[j] = __ballot_sync(0xffffffffu, runs && p + 1 < N && ((w[j] ^ nb) < lim));
        }
        auto left = [&](int j) { return (R[j] << 1) | (j > 0 ? R[j > 0 ? j - 1 : 0] >> 31 : c0); };
        auto valid = [&](int j) {   // lanes whose position is below N
            const long long n = N - (p0 + 32 * j);
            return n >= 32 ? 0xffffffffu : n <= 0 ? 0u : (1u << (int)n) - 1u;
        };
        unsigned nh = 0;
#pragma unroll
        for (int j = 0; j < kFixItems; ++j) {
            const bool alone = ((valid(j) & ~R[j] & ~left(j)) >> lane) & 1u;
            if (alone) {
                const unsigned idx = (unsigned)w[j] & imask;
                P.perm[p0 + 32 * j + lane] = idx;
                if (P.keys_sorted) P.keys_sorted[p0 + 32 * j + lane] = __ldcg(P.keys + idx);   // etics_mex_sort only
            }
            nh += __popc(R[j] & ~left(j));
        }
        if (nh) {   // warp-uniform: one atomic per warp and step
            unsigned at = 0;
            if (lane == 0) at = atomicAdd(&P.hdr->nheads, nh);
            at = __shfl_sync(0xffffffffu, at, 0);
#pragma unroll
            for (int j = 0; j < kFixItems; ++j) {
                const unsigned H = R[j] & ~left(j);   // heads of runs
                if ((H >> lane) & 1u) heads[at + __popc(H & lt_mask)] = (unsigned)(p0 + 32 * j + lane);
                at += __popc(H);
            }
        }
    }
}

// phase F2: one thread per run.
__device__ __forceinline__ void sort_phase_fixruns(const SortParams& P, const SortPlan& pl, const unsigned long long* words,
                                                   const unsigned* heads) {
    const unsigned n = __ldcg(&P.hdr->nheads);
    const unsigned stride = gridDim.x * kSortThreads;
    for (unsigned i = blockIdx.x * kSortThreads + threadIdx.x; i < n; i += stride) {
        const long long p = __ldcg(heads + i);
        sort_fix_run(P, pl, words, p, __ldcg(words + p));
    }
}

// =========================================================================================================
// Fallback: stable LSD sort of (full key, index), eight 8-bit passes, ONE block (histogram by all threads, stable
// scatter by warp 0, 32 keys per step).  Runs only when the fix-up raised the flag.
// =========================================================================================================
__device__ __noinline__ void sort_fallback_block(const unsigned long long* keys, long long N,
                                                 unsigned long long* kA, unsigned long long* kB, unsigned* iA, unsigned* iB,
                                                 unsigned long long* keys_sorted) {
    __shared__ unsigned hist[256];
    __shared__ unsigned base[256];
    __shared__ int single;
    const int nthr = blockDim.x;   // >= 256
    const int tid = threadIdx.x, lane = tid & 31;
    int cur = -1;   // -1: the source is (keys, identity); 0: set A; 1: set B
    for (int pass = 0; pass < 8; ++pass) {
        const int shift = 8 * pass;
        const unsigned long long* ksrc = (cur < 0) ? keys : (cur == 0 ? kA : kB);
        const unsigned* isrc = (cur < 0) ? nullptr : (cur == 0 ? iA : iB);
        unsigned long long* kdst = (cur == 0) ? kB : kA;
        unsigned* idst = (cur == 0) ? iB : iA;
        if (tid < 256) hist[tid] = 0;
        if (tid == 0) single = 0;
        __syncthreads();
        for (long long k = tid; k < N; k += nthr) atomicAdd(&hist[(unsigned)(ksrc[k] >> shift) & 255u], 1u);
        __syncthreads();
        if (tid < 256 && hist[tid] == (unsigned)N) single = 1;
        __syncthreads();
        const bool skip = single != 0 && cur >= 0;   // every key has the same digit: a stable pass would change nothing
        __syncthreads();                              // `single` is rewritten at the top of the next pass
        if (skip) continue;
        if (tid == 0) {
            unsigned run = 0;
            for (int d = 0; d < 256; ++d) { base[d] = run; run += hist[d]; }
        }
        __syncthreads();
        if (tid < 32) {
            for (long long k0 = 0; k0 < N; k0 += 32) {
                const long long k = k0 + lane;
                const bool ok = k < N;
                const unsigned long long key = ok ? ksrc[k] : 0ull;
                const unsigned d = ok ? ((unsigned)(key >> shift) & 255u) : 256u;
                unsigned peers = 0xffffffffu;
#pragma unroll
                for (int b = 0; b < 9; ++b) {
                    const bool bit = (d >> b) & 1u;
                    const unsigned vote = __ballot_sync(0xffffffffu, bit);
                    peers &= bit ? vote : ~vote;
                }
                if (ok) {
                    const unsigned lower = peers & ((1u << lane) - 1u);
                    const unsigned g = base[d] + __popc(lower);
                    kdst[g] = key;
                    idst[g] = isrc ? isrc[k] : (unsigned)k;
                }
                __syncwarp();
                if (ok && (peers & ((1u << lane) - 1u)) == 0u) base[d] += __popc(peers);
                __syncwarp();
            }
        }
        __threadfence();
        __syncthreads();
        cur = (cur == 0) ? 1 : 0;
    }
    // the result belongs in set A (iA is the caller's permutation)
    if (cur == 1) {
        for (long long k = tid; k < N; k += nthr) { kA[k] = kB[k]; iA[k] = iB[k]; }
        __threadfence();
        __syncthreads();
    }
    if (keys_sorted)
        for (long long k = tid; k < N; k += nthr) keys_sorted[k] = kA[k];
}

__global__ void __launch_bounds__(1024)
mex_sort_fallback_kernel(const SortHeader* __restrict__ hdr, const unsigned long long* keys, long long N,
                         unsigned long long* kA, unsigned long long* kB, unsigned* iA, unsigned* iB,
                         unsigned long long* keys_sorted) {
    if (__ldcg(&hdr->fallback) == 0u) return;
    sort_fallback_block(keys, N, kA, kB, iA, iB, keys_sorted);
}

// ---- single-wave sort: every phase in one cooperative launch ---------------------------------------------------
constexpr int kSmallDB = kSortDigitBits;   // 11-bit digits, at most three passes
constexpr int kLargeDB = 9;                // 9-bit digits, at most four passes over 36 prefix bits
constexpr int kLargePrefixBits = 4 * kLargeDB;

#ifdef ETICS_SORT_PROF
#define ETICS_PROF() do { if (blockIdx.x == 0 && threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); P.hdr->prof[prof_i++] = t_; } } while (0)
#else
#define ETICS_PROF() do {} while (0)
#endif

__global__ void __launch_bounds__(kSortThreads, 2)
mex_sort_small_kernel(const __grid_constant__ SortParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem<kSmallDB>& S = *reinterpret_cast<SortSmem<kSmallDB>*>(smem_raw);
    constexpr int BINS = SortSmem<kSmallDB>::BINS;
    cg::grid_group grid = cg::this_grid();
#ifdef ETICS_SORT_PROF
    int prof_i = 0;
#endif
    ETICS_PROF();
    sort_phase_keys(P, S.red);
    ETICS_PROF();
    grid.sync();
    ETICS_PROF();
    const SortPlan pl = load_plan(P.hdr, P.N, P.prefix_bits, P.digit_bits);
    sort_phase_hist<true, kSortTile>(P, S.run, BINS, pl, 0, nullptr);
    ETICS_PROF();
    grid.sync();
    ETICS_PROF();
    for (int pass = 0; pass < pl.passes; ++pass) {   // pl is the same in every block: the barriers match
        const unsigned long long* in = (pass & 1) ? P.bufB : P.bufA;
        unsigned long long* out = (pass & 1) ? P.bufA : P.bufB;
        if (pass > 0) {
            sort_phase_hist<false, kSortTile>(P, S.run, BINS, pl, pass, in);
            ETICS_PROF();
            grid.sync();
            ETICS_PROF();
        }
        sort_phase_scan(P, reinterpret_cast<unsigned*>(S.stage), BINS);
        ETICS_PROF();
        grid.sync();
        ETICS_PROF();
        sort_phase_scatter<kSmallDB, kSortItems>(P, S, pl, pass, in, out);
        ETICS_PROF();
        grid.sync();
        ETICS_PROF();
    }
    const unsigned long long* words = (pl.passes & 1) ? P.bufB : P.bufA;
    unsigned* heads = reinterpret_cast<unsigned*>((pl.passes & 1) ? P.bufA : P.bufB);
    sort_phase_fixup(P, pl, words, heads);
    ETICS_PROF();
    grid.sync();
    sort_phase_fixruns(P, pl, words, heads);
    ETICS_PROF();
    grid.sync();
    if (blockIdx.x == 0 && __ldcg(&P.hdr->fallback) != 0u)   // never taken by the paper's workloads
        sort_fallback_block(P.keys, P.N, P.bufA, P.bufB, P.perm, P.itmp, P.keys_sorted);
}

// ---- bandwidth-bound sort: one kernel per phase; a pass beyond the plan's last one returns at once -----------------
__global__ void __launch_bounds__(kSortThreads)
mex_sort_keys_kernel(const __grid_constant__ SortParams P) {
    __shared__ unsigned long long red[2][kSortWarps];
    sort_phase_keys(P, red);
}

__global__ void __launch_bounds__(kSortThreads)
mex_sort_hist_kernel(const __grid_constant__ SortParams P, int pass) {
    __shared__ unsigned hist[1 << kLargeDB];
    const SortPlan pl = load_plan(P.hdr, P.N, P.prefix_bits, P.digit_bits);
    if (pass > 0 && pass >= pl.passes) return;
    if (pass == 0) sort_phase_hist<true, kSortThreads * kLargeItems>(P, hist, 1 << kLargeDB, pl, 0, nullptr);
    else sort_phase_hist<false, kSortThreads * kLargeItems>(P, hist, 1 << kLargeDB, pl, pass, (pass & 1) ? P.bufB : P.bufA);
}

__global__ void __launch_bounds__(kSortThreads)
mex_sort_scan_kernel(const __grid_constant__ SortParams P, int pass) {
    __shared__ __align__(16) unsigned strip[kSortMaxSegs * kScanStrip];
    const SortPlan pl = load_plan(P.hdr, P.N, P.prefix_bits, P.digit_bits);
    if (pass >= pl.passes) return;
    sort_phase_scan(P, strip, 1 << kLargeDB);
}

using LargeSmem = SortSmem<kLargeDB, kLargeItems>;

__global__ void __launch_bounds__(kSortThreads, kLargeMinBlocks)
mex_sort_scatter_kernel(const __grid_constant__ SortParams P, int pass) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    LargeSmem& S = *reinterpret_cast<LargeSmem*>(smem_raw);
    const SortPlan pl = load_plan(P.hdr, P.N, P.prefix_bits, P.digit_bits);
    if (pass >= pl.passes) return;
    sort_phase_scatter<kLargeDB, kLargeItems>(P, S, pl, pass, (pass & 1) ? P.bufB : P.bufA, (pass & 1) ? P.bufA : P.bufB);
}

__global__ void __launch_bounds__(kSortThreads, 4)
mex_sort_fixup_kernel(const __grid_constant__ SortParams P) {
    const SortPlan pl = load_plan(P.hdr, P.N, P.prefix_bits, P.digit_bits);
    sort_phase_fixup(P, pl, (pl.passes & 1) ? P.bufB : P.bufA, reinterpret_cast<unsigned*>((pl.passes & 1) ? P.bufA : P.bufB));
}

__global__ void __launch_bounds__(kSortThreads)
mex_sort_fixruns_kernel(const __grid_constant__ SortParams P) {
    const SortPlan pl = load_plan(P.hdr, P.N, P.prefix_bits, P.digit_bits);
    sort_phase_fixruns(P, pl, (pl.passes & 1) ? P.bufB : P.bufA, reinterpret_cast<const unsigned*>((pl.passes & 1) ? P.bufA : P.bufB));
}

// ---------------------------------------------------------------------------------------------------------
// Host side.
// ---------------------------------------------------------------------------------------------------------
struct SortDevice { int small_blocks; int scatter_blocks; };   // resident blocks of the cooperative kernel / of the scatter kernel

static cudaError_t sort_device(SortDevice* out) {
    static std::mutex mu;
    static SortDevice cached[64];
    static bool have[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && have[dev]) { *out = cached[dev]; return cudaSuccess; }
    SortDevice d{};
    int per_sm = 0;
    e = cudaFuncSetAttribute(mex_sort_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem<kSmallDB>));
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mex_sort_small_kernel, kSortThreads, sizeof(SortSmem<kSmallDB>));
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    d.small_blocks = device_sm_count() * per_sm;
    if (d.small_blocks > kSortMaxSegs) d.small_blocks = kSortMaxSegs;
    e = cudaFuncSetAttribute(mex_sort_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LargeSmem));
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mex_sort_scatter_kernel, kSortThreads, sizeof(LargeSmem));
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    d.scatter_blocks = device_sm_count() * per_sm;
    if (dev >= 0 && dev < 64) { cached[dev] = d; have[dev] = true; }
    *out = d;
    return cudaSuccess;
}

// kernels one sort launches (for the launch count bench.py reports): the cooperative kernel, or
// keys + (histogram, scan, scatter) per pass + the two fix-up kernels + the fallback kernel
int mex_sort_kernel_launches(long long N) {
    SortDevice dv;
    if (sort_device(&dv) != cudaSuccess) return 0;
    const long long tiles = (N + kSortTile - 1) / kSortTile;
    return tiles <= dv.small_blocks ? 1 : 1 + 3 * (kLargePrefixBits / kLargeDB) + 2 + 1;
}

cudaError_t mex_sort_init_device() {
    SortDevice d;
    return sort_device(&d);
}

cudaError_t mex_sort_enqueue(const double* pos, const double* mass, long long N, const MexLayout& L, char* ws,
                             unsigned* perm_out, unsigned long long* keys_sorted_out, bool pack, cudaStream_t st,
                             cudaEvent_t ev_keygen) {
    SortDevice dv;
    cudaError_t e = sort_device(&dv);
    if (e != cudaSuccess) return e;
    SortParams P{};
    P.pos = pos; P.mass = mass; P.N = N;
    P.keys = reinterpret_cast<unsigned long long*>(ws + L.off_keys);
    P.pk = pack ? reinterpret_cast<double2*>(ws + L.off_pk) : nullptr;
    P.hdr = reinterpret_cast<SortHeader*>(ws + L.off_hdr);
    P.bufA = reinterpret_cast<unsigned long long*>(ws + L.off_wordsA);
    P.bufB = reinterpret_cast<unsigned long long*>(ws + L.off_wordsB);
    P.seg_hist = reinterpret_cast<unsigned*>(ws + L.off_seghist);
    P.bin_tot = reinterpret_cast<unsigned*>(ws + L.off_bintot);
    P.perm = perm_out; P.keys_sorted = keys_sorted_out;
    P.itmp = reinterpret_cast<unsigned*>(ws + L.off_itmp);
    P.tiles = (N + kSortTile - 1) / kSortTile;
    e = cudaMemsetAsync(ws + L.off_hdr, 0, sizeof(SortHeader), st);
    if (e != cudaSuccess) return e;
    if (P.tiles <= dv.small_blocks) {
        // One tile per block: the whole sort is a single wave and latency-bound.  Everything in one cooperative launch,
        // three passes of 11-bit digits.
        P.tps = 1;
        P.nseg = (int)P.tiles;
        P.prefix_bits = kSortPrefixBits;
        P.digit_bits = kSmallDB;
        void* args[] = {&P};
        int grid = (int)P.tiles < 128 ? 128 : (int)P.tiles;   // fewer blocks: cheaper grid barriers
        if (grid > dv.small_blocks) grid = dv.small_blocks;
        e = cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(mex_sort_small_kernel), dim3((unsigned)grid),
                                        dim3(kSortThreads), args, sizeof(SortSmem<kSmallDB>), st);
        if (e != cudaSuccess) return e;
        if (ev_keygen) cudaEventRecord(ev_keygen, st);
        return cudaSuccess;   // the fallback sort is the kernel's last phase
    } else {
        // Bandwidth-bound: one kernel per phase, a block per segment of consecutive tiles (two waves of segments), four
        // passes of 9-bit digits over 36 prefix bits — with 2048 digit values a tile of 4096 words would scatter runs of
        // two words (N = 1e8: 1.41 ms per scatter against 0.66 ms), and fewer prefix bits leave more runs to the fix-up.
        constexpr int kLargeTile = kSortThreads * kLargeItems;
        P.tiles = (N + kLargeTile - 1) / kLargeTile;
        long long segs = 2ll * dv.scatter_blocks;   // two waves of segments (N = 1e8: one wave 4.95 ms, two 4.77, three 4.81)
        if (segs > kSortMaxSegs) segs = kSortMaxSegs;
        P.tps = (P.tiles + segs - 1) / segs;
        P.nseg = (int)((P.tiles + P.tps - 1) / P.tps);
        P.prefix_bits = kLargePrefixBits;
        P.digit_bits = kLargeDB;
        const int wide = device_sm_count() * 8;
        mex_sort_keys_kernel<<<wide, kSortThreads, 0, st>>>(P);
        constexpr int kPasses = kLargePrefixBits / kLargeDB;
        for (int pass = 0; pass < kPasses; ++pass) {
            mex_sort_hist_kernel<<<P.nseg, kSortThreads, 0, st>>>(P, pass);
            mex_sort_scan_kernel<<<(1 << kLargeDB) / kScanStrip, kSortThreads, 0, st>>>(P, pass);
            mex_sort_scatter_kernel<<<P.nseg, kSortThreads, sizeof(LargeSmem), st>>>(P, pass);
        }
        mex_sort_fixup_kernel<<<wide, kSortThreads, 0, st>>>(P);
        mex_sort_fixruns_kernel<<<wide, kSortThreads, 0, st>>>(P);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (ev_keygen) cudaEventRecord(ev_keygen, st);
    mex_sort_fallback_kernel<<<1, 1024, 0, st>>>(P.hdr, P.keys, N, P.bufA, P.bufB, perm_out, P.itmp, keys_sorted_out);
    return cudaGetLastError();
}

}  // namespace etics

// mex_sort.cu — MEX steps M1–M2: radial sort of the particles by r^2 (§3.2: "the
// distance square ... for the sorting operation"), stable, ties broken by particle index.  Hand-written for
// sm_100a, no CUB/Thrust.
//
// The paper sorts whole particle structs with Thrust's merge sort.  Here the sort moves ONE 64-bit
// word per particle and makes at most three passes:
//
//   mex_keygen_kernel   key_k = bits(r_k^2), rounding pinned (t = x*x; t = fma(y,y,t); t = fma(z,z,t)); the
//                       (x,y,z,m) record of the particle as one 32-byte sector; min and max key of the set.
//   mex_pack_kernel     word_k = (prefix_k << ibits) | k, prefix_k = (key_k - kmin) >> shift: the leading
//                       B = min(33, bits(kmax - kmin)) bits of the key's offset from the smallest key, above the
//                       ibits = bits(N-1) bits of the particle index; digit histograms of all passes.
//   mex_radix_pass_kernel  one stable LSD pass over a digit of <= 11 bits of the prefix ("onesweep": ranks inside
//                       the tile, decoupled look-back over the preceding tiles' digit counts — integers, so the
//                       result does not depend on timing — one coalesced write).  The index bits ride along.
//   mex_fixup_kernel    particles whose prefixes collide (the key bits below `shift` were not sorted) form short runs;
//                       the thread at the head of a run orders it by (full key, index).  For smooth particle
//                       distributions a fraction ~N / 2^27 per octave of r^2 collides.  shift = 0: nothing to do.
//   mex_sort_fallback_kernel   a run longer than kFixMaxRun (many particles within 2^shift ulps of each other, yet
//                       not all equal: e.g. two thin shells) raises a flag and this plain single-block LSD sort
//                       of the full keys redoes the job — correct for any input, slow, never taken by the paper's workloads.
//
// Why 33 bits: an r^2 range of 44 octaves (r from 1e-4 to 300) needs 6 exponent bits, which leaves 27 mantissa bits
// in the prefix; three 11-bit passes over 8-byte words move 48 bytes per particle where eight 8-bit passes over
// (key, index) pairs moved 192.
#include "mex_common.cuh"

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

__host__ __device__ inline SortPlan make_sort_plan(unsigned long long kmin, unsigned long long kmax, long long N) {
    SortPlan p;
    p.kmin = kmin;
    p.ibits = bit_length64((unsigned long long)(N - 1));
    const int nbits = bit_length64(kmax - kmin);
    p.B = nbits < kSortPrefixBits ? nbits : kSortPrefixBits;
    p.shift = nbits - p.B;
    p.passes = (p.B + kSortDigitBits - 1) / kSortDigitBits;
    return p;
}

__device__ __forceinline__ SortPlan load_plan(const SortHeader* hdr, long long N) {
    const unsigned long long inv = __ldcg(&hdr->inv_kmin), kmax = __ldcg(&hdr->kmax);
    return make_sort_plan(~inv, kmax, N);
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

constexpr int kKeygenItems = 4;

// PACK: also write (x, y, z, m) of particle k as one 32-byte record pk[k], so that the gather after the sort reads
// one aligned sector per particle instead of four.
template <bool PACK>
__global__ void __launch_bounds__(256)
mex_keygen_kernel(const double* __restrict__ pos, const double* __restrict__ mass, long long N,
                  unsigned long long* __restrict__ keys, double2* __restrict__ pk, SortHeader* __restrict__ hdr) {
    __shared__ unsigned long long s_inv[8], s_max[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long inv = 0, mx = 0;
    const long long stride = (long long)gridDim.x * 256 * kKeygenItems;
    for (long long base = (long long)blockIdx.x * 256 * kKeygenItems; base < N; base += stride) {
        double x[kKeygenItems], y[kKeygenItems], z[kKeygenItems], mk[kKeygenItems];
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * 256 + threadIdx.x;
            const bool ok = k < N;
            x[j] = ok ? pos[k] : 0.0; y[j] = ok ? pos[N + k] : 0.0; z[j] = ok ? pos[2 * N + k] : 0.0;
            if (PACK) mk[j] = ok ? mass[k] : 0.0;
        }
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * 256 + threadIdx.x;
            if (k < N) {
                const unsigned long long key = mex_key(x[j], y[j], z[j]);
                keys[k] = key;
                if (PACK) { pk[2 * k] = make_double2(x[j], y[j]); pk[2 * k + 1] = make_double2(z[j], mk[j]); }
                inv = max(inv, ~key);
                mx = max(mx, key);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        inv = max(inv, __shfl_xor_sync(0xffffffffu, inv, o));
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if (lane == 0) { s_inv[warp] = inv; s_max[warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < 8; ++w) { inv = max(inv, s_inv[w]); mx = max(mx, s_max[w]); }
        atomicMax(&hdr->inv_kmin, inv);   // integer atomics: the result does not depend on their order
        atomicMax(&hdr->kmax, mx);
    }
}

// =========================================================================================================
// Packed words and the digit histograms of every pass.
// =========================================================================================================
__global__ void __launch_bounds__(256)
mex_pack_kernel(const unsigned long long* __restrict__ keys, long long N, const SortHeader* __restrict__ hdr,
                unsigned long long* __restrict__ words, unsigned* __restrict__ hist) {
    __shared__ unsigned sh[kSortMaxPasses * kSortBins];
    const SortPlan pl = load_plan(hdr, N);
    for (int i = threadIdx.x; i < kSortMaxPasses * kSortBins; i += 256) sh[i] = 0;
    __syncthreads();
    const long long stride = (long long)gridDim.x * 256 * kKeygenItems;
    for (long long base = (long long)blockIdx.x * 256 * kKeygenItems; base < N; base += stride) {
        unsigned long long key[kKeygenItems];
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * 256 + threadIdx.x;
            key[j] = (k < N) ? keys[k] : 0ull;
        }
#pragma unroll
        for (int j = 0; j < kKeygenItems; ++j) {
            const long long k = base + j * 256 + threadIdx.x;
            if (k < N) {
                const unsigned long long pre = (key[j] - pl.kmin) >> pl.shift;
                words[k] = (pre << pl.ibits) | (unsigned long long)k;
#pragma unroll
                for (int p = 0; p < kSortMaxPasses; ++p)
                    if (p < pl.passes) atomicAdd(&sh[p * kSortBins + (unsigned)((pre >> pl.lo(p)) & ((1u << pl.w(p)) - 1u))], 1u);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kSortMaxPasses * kSortBins; i += 256)
        if (sh[i]) atomicAdd(&hist[i], sh[i]);
}

// =========================================================================================================
// M2: one stable LSD radix pass with decoupled look-back.
//
// Tile = 256 threads x ITEMS words, loaded warp-striped (item i of warp w at tile base + w*32*ITEMS + 32 i + lane), so the
// order (warp, item, lane) is the order of the input.
// Ranking: per warp and digit a 16-bit counter [tag:5 | count:11].  For every item the lanes stamp their lane
// number on their digit's counter and read it back: if every lane finds its own stamp, all 32 digits of the item
// are distinct (78 % of the items for uniformly distributed 11-bit digits) and the rank is simply the counter;
// otherwise the lanes that share a digit find each other with one ballot per digit bit.  (Measured in round 1:
// MATCH.ANY iterates over the distinct values of a warp, ~230 cycles for random digits; shared-memory atomics do
// not return ranks in lane order.)
// Status word of (tile, digit): bit 31 = inclusive prefix (31-bit count), else bit 30 = tile aggregate, else not yet
// posted.  One status array per pass, zeroed with the header.
// Launched with programmatic stream serialisation: the prologue (ticket, clearing the counters) overlaps the tail
// of the preceding kernel; griddepcontrol.wait orders every read of its output, and those reads are L2-coherent.
// =========================================================================================================
constexpr unsigned kFlagIncl = 0x80000000u, kFlagAgg = 0x40000000u;
constexpr int kBinsPerThread = kSortBins / kSortThreads;   // 8: thread t owns digits 8t..8t+7 in the offset phases
constexpr int kLookW = 2;                                  // status rows in flight per look-back round
static_assert(kBinsPerThread == 8, "the offset phases move the eight 16-bit counters of a thread as one 16-byte vector");

template <int ITEMS>
struct SortSmem {
    unsigned short cnt[kSortWarps][kSortBins];   // ranking: [tag | count]; afterwards position of (warp, digit) inside the tile
    unsigned gbase[kSortBins];                   // global position of the tile's first word of digit d, minus its tile position
    unsigned scan_tmp[kSortWarps];
    unsigned tile;
    unsigned long long stage[kSortThreads * ITEMS];
};

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ uint4 ld_volatile_v4(const unsigned* p) {
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_v4(unsigned* p, uint4 v) {
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

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
    __syncthreads();
    return woff + inc - v;
}

template <int ITEMS, int MINB>
__global__ void __launch_bounds__(kSortThreads, MINB)
mex_radix_pass_kernel(const unsigned long long* __restrict__ bufA, unsigned long long* __restrict__ bufB,
                      long long N, int pass, SortHeader* __restrict__ hdr, const unsigned* __restrict__ hist,
                      unsigned* status_all, long long status_rows) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem<ITEMS>& S = *reinterpret_cast<SortSmem<ITEMS>*>(smem_raw);
    constexpr int TILE = kSortThreads * ITEMS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    pdl_launch_dependents();
    if (tid == 0) S.tile = atomicAdd(&hdr->tickets[pass], 1u);   // tiles are numbered in the order they start running
    {
        uint4* c = reinterpret_cast<uint4*>(&S.cnt[0][0]);
        constexpr int kVec = kSortWarps * kSortBins * 2 / 16;
#pragma unroll
        for (int i = 0; i < kVec / kSortThreads; ++i) c[i * kSortThreads + tid] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    const long long tile = S.tile;
    pdl_wait();

    const SortPlan pl = load_plan(hdr, N);
    if (pass >= pl.passes) return;   // fewer digits than passes: the data stays where it is
    const unsigned long long* __restrict__ in = (pass & 1) ? bufB : bufA;
    unsigned long long* __restrict__ out = (pass & 1) ? const_cast<unsigned long long*>(bufA) : bufB;
    const int dshift = pl.ibits + pl.lo(pass);
    const unsigned dmask = (1u << pl.w(pass)) - 1u;
    unsigned* status = status_all + (size_t)pass * status_rows * kSortBins;

    // ---- load ---------------------------------------------------------------------------------------------
    const long long base = tile * TILE + (long long)warp * (32 * ITEMS);
    unsigned long long key[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const long long k = base + 32 * i + lane;
        key[i] = (k < N) ? __ldcg(in + k) : ~0ull;   // padding sorts last in every pass and is never written (position >= N)
    }
    // global start of every bucket: exclusive scan of the pass's histogram
    unsigned hb[kBinsPerThread];
    {
        const uint4 h0 = __ldcg(reinterpret_cast<const uint4*>(hist + pass * kSortBins + kBinsPerThread * tid));
        const uint4 h1 = __ldcg(reinterpret_cast<const uint4*>(hist + pass * kSortBins + kBinsPerThread * tid) + 1);
        hb[0] = h0.x; hb[1] = h0.y; hb[2] = h0.z; hb[3] = h0.w; hb[4] = h1.x; hb[5] = h1.y; hb[6] = h1.z; hb[7] = h1.w;
        unsigned run = 0;
#pragma unroll
        for (int q = 0; q < kBinsPerThread; ++q) { const unsigned t = hb[q]; hb[q] = run; run += t; }
        const unsigned off = block_exclusive_scan_256(run, S.scan_tmp);
#pragma unroll
        for (int q = 0; q < kBinsPerThread; ++q) hb[q] += off;
    }

    // ---- rank ---------------------------------------------------------------------------------------------
    unsigned short rank[ITEMS];
    volatile unsigned short* cw = S.cnt[warp];
    const unsigned lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
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
            for (int b = 0; b < kSortDigitBits; ++b) {
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
    __syncthreads();

    // ---- thread t owns digits 8t..8t+7: per-warp counts -> exclusive over warps, tile totals -----------------
    unsigned tot[kBinsPerThread];
    {
        uint4 run = make_uint4(0u, 0u, 0u, 0u);   // eight 16-bit running sums, two per word (<= TILE < 65536)
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            uint4* p = reinterpret_cast<uint4*>(&S.cnt[w][kBinsPerThread * tid]);
            uint4 v = *p;
            v.x &= 0x07ff07ffu; v.y &= 0x07ff07ffu; v.z &= 0x07ff07ffu; v.w &= 0x07ff07ffu;
            *p = run;
            run.x += v.x; run.y += v.y; run.z += v.z; run.w += v.w;
        }
        tot[0] = run.x & 0xffffu; tot[1] = run.x >> 16; tot[2] = run.y & 0xffffu; tot[3] = run.y >> 16;
        tot[4] = run.z & 0xffffu; tot[5] = run.z >> 16; tot[6] = run.w & 0xffffu; tot[7] = run.w >> 16;
    }
    unsigned* my_status = status + (size_t)tile * kSortBins + kBinsPerThread * tid;
    {
        const unsigned f = (tile > 0) ? kFlagAgg : kFlagIncl;   // tile 0: its totals are its inclusive prefixes
        st_volatile_v4(my_status, make_uint4(f | tot[0], f | tot[1], f | tot[2], f | tot[3]));
        st_volatile_v4(my_status + 4, make_uint4(f | tot[4], f | tot[5], f | tot[6], f | tot[7]));
    }
    unsigned loc[kBinsPerThread];   // position of the tile's first word of digit d inside the tile
    {
        unsigned run = 0;
#pragma unroll
        for (int q = 0; q < kBinsPerThread; ++q) { loc[q] = run; run += tot[q]; }
        const unsigned off = block_exclusive_scan_256(run, S.scan_tmp);
#pragma unroll
        for (int q = 0; q < kBinsPerThread; ++q) loc[q] += off;
        const uint4 add = make_uint4(loc[0] | (loc[1] << 16), loc[2] | (loc[3] << 16), loc[4] | (loc[5] << 16), loc[6] | (loc[7] << 16));
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            uint4* p = reinterpret_cast<uint4*>(&S.cnt[w][kBinsPerThread * tid]);
            uint4 v = *p;
            v.x += add.x; v.y += add.y; v.z += add.z; v.w += add.w;
            *p = v;
        }
    }
    __syncthreads();

    // ---- reorder inside the tile (stable); the words leave the registers before the look-back -------------------
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const unsigned d = (unsigned)(key[i] >> dshift) & dmask;
        S.stage[S.cnt[warp][d] + rank[i]] = key[i];
    }

    // ---- decoupled look-back over the preceding tiles, kLookW status rows in flight ------------------------------
    unsigned excl[kBinsPerThread];
#pragma unroll
    for (int q = 0; q < kBinsPerThread; ++q) excl[q] = 0u;
    if (tile > 0) {
        unsigned pending = 0xffu;
        long long t = tile - 1;
        while (pending) {
            uint4 a[kLookW], b[kLookW];
#pragma unroll
            for (int j = 0; j < kLookW; ++j) {
                const long long tt = (t - j >= 0) ? t - j : 0;   // rows before tile 0 are never consumed (tile 0 posts inclusive prefixes)
                const unsigned* row = status + (size_t)tt * kSortBins + kBinsPerThread * tid;
                a[j] = ld_volatile_v4(row);
                b[j] = ld_volatile_v4(row + 4);
            }
            int used = 0;
#pragma unroll
            for (int j = 0; j < kLookW; ++j) {
                if (pending && used == j) {
                    const unsigned v[kBinsPerThread] = {a[j].x, a[j].y, a[j].z, a[j].w, b[j].x, b[j].y, b[j].z, b[j].w};
                    bool ready = true;
#pragma unroll
                    for (int q = 0; q < kBinsPerThread; ++q) ready = ready && (((pending >> q) & 1u) == 0u || (v[q] >> 30) != 0u);
                    if (ready) {
#pragma unroll
                        for (int q = 0; q < kBinsPerThread; ++q) {
                            if ((pending >> q) & 1u) {
                                if (v[q] & kFlagIncl) { excl[q] += v[q] & 0x7fffffffu; pending &= ~(1u << q); }
                                else excl[q] += v[q] & 0x3fffffffu;
                            }
                        }
                        used = j + 1;
                    }
                }
            }
            t -= used;
            if (used == 0) __nanosleep(32);
        }
    }
    if (tile > 0) {
        st_volatile_v4(my_status, make_uint4(kFlagIncl | (excl[0] + tot[0]), kFlagIncl | (excl[1] + tot[1]),
                                             kFlagIncl | (excl[2] + tot[2]), kFlagIncl | (excl[3] + tot[3])));
        st_volatile_v4(my_status + 4, make_uint4(kFlagIncl | (excl[4] + tot[4]), kFlagIncl | (excl[5] + tot[5]),
                                                 kFlagIncl | (excl[6] + tot[6]), kFlagIncl | (excl[7] + tot[7])));
    }
    {
        uint4* gb = reinterpret_cast<uint4*>(&S.gbase[kBinsPerThread * tid]);
        gb[0] = make_uint4(hb[0] + excl[0] - loc[0], hb[1] + excl[1] - loc[1], hb[2] + excl[2] - loc[2], hb[3] + excl[3] - loc[3]);
        gb[1] = make_uint4(hb[4] + excl[4] - loc[4], hb[5] + excl[5] - loc[5], hb[6] + excl[6] - loc[6], hb[7] + excl[7] - loc[7]);
    }
    __syncthreads();

    // ---- write runs of equal digits -------------------------------------------------------------------------------
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
        const unsigned j = i * kSortThreads + tid;
        const unsigned long long kk = S.stage[j];
        const unsigned d = (unsigned)(kk >> dshift) & dmask;
        const unsigned g = S.gbase[d] + j;
        if ((long long)g < N) out[g] = kk;
    }
}

// =========================================================================================================
// Fix-up: order the runs of equal prefixes by (full key, index); write the permutation (and the sorted keys).
// =========================================================================================================
constexpr int kFixMaxRun = 32;

__global__ void __launch_bounds__(256)
mex_fixup_kernel(const unsigned long long* __restrict__ bufA, const unsigned long long* __restrict__ bufB,
                 const unsigned long long* __restrict__ keys, long long N, SortHeader* __restrict__ hdr,
                 unsigned* __restrict__ perm, unsigned long long* __restrict__ keys_sorted) {
    const SortPlan pl = load_plan(hdr, N);
    const unsigned long long* __restrict__ words = (pl.passes & 1) ? bufB : bufA;
    const unsigned long long imask = (pl.ibits >= 64) ? ~0ull : ((1ull << pl.ibits) - 1ull);
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const unsigned long long w = words[p];
    const unsigned long long pre = w >> pl.ibits;
    const bool run_left = pl.shift > 0 && p > 0 && (words[p - 1] >> pl.ibits) == pre;
    const bool run_right = pl.shift > 0 && p + 1 < N && (words[p + 1] >> pl.ibits) == pre;
    if (!run_left && !run_right) {
        const unsigned i = (unsigned)(w & imask);
        perm[p] = i;
        if (keys_sorted) keys_sorted[p] = keys[i];
        return;
    }
    if (run_left) return;   // the head of the run writes for all its members
    unsigned idx[kFixMaxRun];
    unsigned long long key[kFixMaxRun];
    int len = 0;
    while (p + len < N && len < kFixMaxRun) {
        const unsigned long long v = (len == 0) ? w : words[p + len];
        if ((v >> pl.ibits) != pre) break;
        idx[len] = (unsigned)(v & imask);
        ++len;
    }
    if (len == kFixMaxRun && p + len < N && (words[p + len] >> pl.ibits) == pre) {
        atomicExch(&hdr->fallback, 1u);   // too long to order here: the fallback sort redoes the whole job
        return;
    }
    for (int j = 0; j < len; ++j) key[j] = keys[idx[j]];
    // stable insertion sort by the full key: members arrive in index order (the passes are stable)
    for (int j = 1; j < len; ++j) {
        const unsigned long long kj = key[j];
        const unsigned ij = idx[j];
        int q = j - 1;
        while (q >= 0 && key[q] > kj) { key[q + 1] = key[q]; idx[q + 1] = idx[q]; --q; }
        key[q + 1] = kj; idx[q + 1] = ij;
    }
    for (int j = 0; j < len; ++j) {
        perm[p + j] = idx[j];
        if (keys_sorted) keys_sorted[p + j] = key[j];
    }
}

// =========================================================================================================
// Fallback: stable LSD sort of (full key, index), eight 8-bit passes, ONE block (histogram by all threads, stable
// scatter by warp 0, 32 keys per step).  Runs only when the fix-up raised the flag.
// =========================================================================================================
__global__ void __launch_bounds__(1024)
mex_sort_fallback_kernel(const SortHeader* __restrict__ hdr, const unsigned long long* __restrict__ keys, long long N,
                         unsigned long long* kA, unsigned long long* kB, unsigned* iA, unsigned* iB,
                         unsigned long long* keys_sorted) {
    if (__ldcg(&hdr->fallback) == 0u) return;
    __shared__ unsigned hist[256];
    __shared__ unsigned base[256];
    __shared__ int single;
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
        for (long long k = tid; k < N; k += 1024) atomicAdd(&hist[(unsigned)(ksrc[k] >> shift) & 255u], 1u);
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
        for (long long k = tid; k < N; k += 1024) { kA[k] = kB[k]; iA[k] = iB[k]; }
        __threadfence();
        __syncthreads();
    }
    if (keys_sorted)
        for (long long k = tid; k < N; k += 1024) keys_sorted[k] = kA[k];
}

// ---------------------------------------------------------------------------------------------------------
// Host side.
// ---------------------------------------------------------------------------------------------------------
constexpr long long kSortSmallN = 1ll << 22;   // below: 4096-word tiles (more tiles in flight); above: 8192-word tiles

template <int ITEMS, int MINB>
static cudaError_t radix_pass_set_attr() {
    return cudaFuncSetAttribute(mex_radix_pass_kernel<ITEMS, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)sizeof(SortSmem<ITEMS>));
}

cudaError_t mex_sort_init_device() {
    static DeviceOnce once;
    return once.run([] {
        cudaError_t e = radix_pass_set_attr<16, 3>();
        if (e != cudaSuccess) return e;
        return radix_pass_set_attr<32, 2>();
    });
}

template <int ITEMS, int MINB>
static cudaError_t radix_passes_enqueue(unsigned long long* bufA, unsigned long long* bufB, long long N, SortHeader* hdr,
                                        const unsigned* hist, unsigned* status, long long status_rows, cudaStream_t st) {
    auto kern = mex_radix_pass_kernel<ITEMS, MINB>;
    constexpr int TILE = kSortThreads * ITEMS;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)((N + TILE - 1) / TILE));
    cfg.blockDim = dim3(kSortThreads);
    cfg.dynamicSmemBytes = sizeof(SortSmem<ITEMS>);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    for (int pass = 0; pass < kSortMaxPasses; ++pass) {
        cudaError_t e = cudaLaunchKernelEx(&cfg, kern, (const unsigned long long*)bufA, bufB, N, pass, hdr, hist, status, status_rows);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t mex_sort_enqueue(const double* pos, const double* mass, long long N, const MexLayout& L, char* ws,
                             unsigned* perm_out, unsigned long long* keys_sorted_out, bool pack, cudaStream_t st,
                             cudaEvent_t ev_keygen) {
    cudaError_t e = mex_sort_init_device();
    if (e != cudaSuccess) return e;
    SortHeader* hdr = reinterpret_cast<SortHeader*>(ws + L.off_hdr);
    unsigned* hist = reinterpret_cast<unsigned*>(ws + L.off_hist);
    unsigned* status = reinterpret_cast<unsigned*>(ws + L.off_status);
    unsigned long long* keys = reinterpret_cast<unsigned long long*>(ws + L.off_keys);
    unsigned long long* bufA = reinterpret_cast<unsigned long long*>(ws + L.off_wordsA);
    unsigned long long* bufB = reinterpret_cast<unsigned long long*>(ws + L.off_wordsB);
    unsigned* itmp = reinterpret_cast<unsigned*>(ws + L.off_itmp);
    double2* pk = reinterpret_cast<double2*>(ws + L.off_pk);

    e = cudaMemsetAsync(ws + L.off_zero, 0, L.zero_bytes, st);
    if (e != cudaSuccess) return e;
    const long long per_block = 256 * kKeygenItems;
    long long blocks = (N + per_block - 1) / per_block;
    const long long cap = (long long)device_sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (pack) mex_keygen_kernel<true><<<(unsigned)blocks, 256, 0, st>>>(pos, mass, N, keys, pk, hdr);
    else mex_keygen_kernel<false><<<(unsigned)blocks, 256, 0, st>>>(pos, nullptr, N, keys, nullptr, hdr);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    mex_pack_kernel<<<(unsigned)blocks, 256, 0, st>>>(keys, N, hdr, bufA, hist);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (ev_keygen) cudaEventRecord(ev_keygen, st);
    if (N < kSortSmallN) e = radix_passes_enqueue<16, 3>(bufA, bufB, N, hdr, hist, status, L.sort_rows, st);
    else e = radix_passes_enqueue<32, 2>(bufA, bufB, N, hdr, hist, status, L.sort_rows, st);
    if (e != cudaSuccess) return e;
    mex_fixup_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(bufA, bufB, keys, N, hdr, perm_out, keys_sorted_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    mex_sort_fallback_kernel<<<1, 1024, 0, st>>>(hdr, keys, N, bufA, bufB, perm_out, itmp, keys_sorted_out);
    return cudaGetLastError();
}

}  // namespace etics

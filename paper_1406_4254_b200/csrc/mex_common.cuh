// mex_common.cuh — workspace layout and launch plumbing shared by the MEX translation units (mex_sort.cu: M1–M2,
// mex.cu: M3–M7).  Never included by oracle/.
#pragma once

#include "etics_common.cuh"

namespace etics {

// ---- sort geometry (mex_sort.cu) ---------------------------------------------------------------------------
constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortDigitBits = 11;                 // widest digit of a pass
constexpr int kSortBins = 1 << kSortDigitBits;     // 2048
constexpr int kSortMaxPasses = 3;
constexpr int kSortPrefixBits = kSortDigitBits * kSortMaxPasses;   // single-wave sort: 33 key bits are radix-sorted, the rest is fixed up
constexpr int kSortMinTile = kSortThreads * 16;    // words per sort tile
constexpr int kSortMaxSegs = 1024;                 // blocks of the persistent sort kernel (segment histogram rows)

// Header of the sort, in the zeroed part of the workspace.
struct SortHeader {
    unsigned long long inv_kmin;   // max over ~key (so that zero-initialisation works); kmin = ~inv_kmin
    unsigned long long kmax;
    unsigned fallback;             // set by the fix-up when a run of equal prefixes is too long to fix locally
    unsigned nheads;               // runs of equal prefixes listed by the fix-up
    unsigned pad[10];
#ifdef ETICS_SORT_PROF
    unsigned long long prof[32];   // development: %globaltimer of block 0 at the phase boundaries
#endif
};

// ---- scan geometry (mex.cu) --------------------------------------------------------------------------------
constexpr int kMexThreads = 32;          // a scan tile is one warp: lane = chunk of kMexK consecutive sorted particles
#ifndef ETICS_MEX_K
#define ETICS_MEX_K 8
#endif
constexpr int kMexK = ETICS_MEX_K;
constexpr int kMexTile = kMexThreads * kMexK;
constexpr int kRecFields = 8;            // r, 1/r, cos th, sin th, cos ph, sin ph, mass, (spare)

struct MexLayout {
    long long N;
    int lmax;
    long long tiles, chunks;    // scan tiles; chunks = tiles * kMexThreads
    int rows;                   // running sums per particle: 2 directions x (cos,sin) x (l,m)
    size_t off_hdr;             // SortHeader (zeroed by every call)
    size_t off_seghist;         // digit histogram of every sort segment, kSortMaxSegs x kSortBins u32
    size_t off_bintot;          // digit totals, kSortBins u32
    size_t off_keys;            // fp64 bit patterns of r^2 by original index (8N)
    size_t off_wordsA, off_wordsB;   // packed (key prefix | index) words (8N each)
    size_t off_perm;            // sorted order: perm[rank] = original index (4N)
    size_t off_itmp;            // second index buffer of the fallback sort (4N)
    size_t off_pk;              // (x, y, z, m) by original index, one 32-byte sector per particle; later the (Phi, a) records
    size_t off_rec, off_idxT, off_tot;
    size_t total;
};

MexLayout make_mex_layout(long long N, int lmax);   // mex.cu part 0

// mex_sort.cu: M1–M2.  perm_out[rank] = original index; keys_sorted_out may be null; pack: also write the (x,y,z,m)
// records at L.off_pk.  ev_keygen (optional) is recorded after the key generation.
cudaError_t mex_sort_enqueue(const double* pos, const double* mass, long long N, const MexLayout& L, char* ws,
                             unsigned* perm_out, unsigned long long* keys_sorted_out, bool pack, cudaStream_t st,
                             cudaEvent_t ev_keygen);
cudaError_t mex_sort_init_device();
int mex_sort_kernel_launches(long long N);

}  // namespace etics

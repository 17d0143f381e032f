// scf_static.cu — etics_scf_coeffs_static: the SCF coefficients (PAPER.md:217-219 step 1, eq. 18) for callers that cannot
// allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// etics_scf_coeffs keeps its block partials (one table of 2 T sums per accumulation block, at most 148 blocks) in a
// workspace the caller allocates.  Here the same two kernels (scf_accumulate_kernel, scf_finalize_kernel: scf.cu) get
// that workspace from a file-scope __device__ array instead: no cudaMalloc, no cudaFree, no allocating library routine.
//
//   limit     T = (nmax+1) (lmax+1) (lmax+2) / 2  <=  ETICS_STATIC_MAX_TABLE = 1386  (the paper's largest expansion,
//             nmax = 20, lmax = 10; PAPER.md:340 uses (10,6)): 148 x 2 x 1386 x 8 B = 3 282 048 bytes (3.13 MiB).  Every GPU that
//             loads the library holds these bytes until the process exits.  Beyond the limit: ETICS_ERR_STATIC_LIMIT.
//   sharing   every call on a device uses the SAME array.  Calls that overlap on the GPU (different streams, or graphs
//             replayed concurrently) race on it; calls on one stream, or otherwise ordered, are safe.  The array keeps the
//             last call's partials; nothing has to start at zero: every block of the accumulation writes its whole
//             partial table before the finalize kernel reads exactly the tables of this call's blocks.
//
// In host code the name g_scf_scratch is a host-side stand-in for the symbol, not a device address: the address comes
// from cudaGetSymbolAddress, once per device with that device current (DeviceOnce), and only that pointer is handed
// to the launchers.
#include "etics_common.cuh"

namespace etics {

// 148 block partials of 2 T doubles, rounded up to the 256-byte granule of etics_workspace_bytes
constexpr size_t kStaticScratchBytes = ((size_t)148 * 2 * ETICS_STATIC_MAX_TABLE * sizeof(double) + 255) / 256 * 256;

static __device__ __align__(256) unsigned char g_scf_scratch[kStaticScratchBytes];

// device address of g_scf_scratch on the current device (one process may drive several GPUs: each has its own copy)
static cudaError_t static_scratch(void** out) {
    static DeviceOnce once;
    static void* addr[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaGetSymbolAddress(out, g_scf_scratch);
    e = once.run([dev] {
        void* p = nullptr;
        const cudaError_t s = cudaGetSymbolAddress(&p, g_scf_scratch);
        if (s == cudaSuccess) addr[dev] = p;
        return s;
    });
    if (e != cudaSuccess) return e;
    *out = addr[dev];
    return *out ? cudaSuccess : cudaErrorInvalidSymbol;
}

}  // namespace etics

using namespace etics;

extern "C" {

size_t etics_scf_coeffs_static_max_table(void) { return ETICS_STATIC_MAX_TABLE; }

etics_status etics_scf_coeffs_static(const double* pos, const double* mass, long long N, int nmax, int lmax,
                                     double* A, double* B, void* stream) {
    if (N < 1 || N >= (1LL << 31) || nmax < 0 || lmax < 0) return ETICS_ERR_ARG;
    if (nmax > ETICS_MAX_NMAX || lmax > ETICS_MAX_LMAX) return ETICS_ERR_LIMIT;
    if ((size_t)(nmax + 1) * num_lm(lmax) > (size_t)ETICS_STATIC_MAX_TABLE) return ETICS_ERR_STATIC_LIMIT;
    if (scf_coeffs_workspace(N, nmax, lmax) > kStaticScratchBytes) return ETICS_ERR_STATIC_LIMIT;
    if (!pos || !mass || !A || !B) return ETICS_ERR_ARG;
    for (const void* p : {(const void*)pos, (const void*)mass, (const void*)A, (const void*)B})
        if (reinterpret_cast<uintptr_t>(p) & 15u) return ETICS_ERR_ALIGN;
    void* ws = nullptr;
    if (static_scratch(&ws) != cudaSuccess) return ETICS_ERR_CUDA;
    return scf_coeffs_launch(pos, mass, N, nmax, lmax, A, B, ws, static_cast<cudaStream_t>(stream)) == cudaSuccess
               ? ETICS_OK : ETICS_ERR_CUDA;
}

}  // extern "C"

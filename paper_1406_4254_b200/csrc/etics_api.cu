// etics_api.cu — the C ABI of include/etics.h: argument checks, workspace sizes, launch sequences.
// Nothing here computes; every step of the path runs in the kernels of scf.cu / mex.cu.
#include "etics_common.cuh"

using namespace etics;

namespace {

inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

etics_status check_sizes(long long N, int nmax, int lmax) {
    if (N < 1 || N >= (1LL << 31) || nmax < 0 || lmax < 0) return ETICS_ERR_ARG;
    if (nmax > ETICS_MAX_NMAX || lmax > ETICS_MAX_LMAX) return ETICS_ERR_LIMIT;
    return ETICS_OK;
}

inline etics_status from_cuda(cudaError_t e) { return e == cudaSuccess ? ETICS_OK : ETICS_ERR_CUDA; }

}  // namespace

extern "C" {

const char* etics_status_string(etics_status s) {
    switch (s) {
        case ETICS_OK: return "ETICS_OK";
        case ETICS_ERR_ARG: return "ETICS_ERR_ARG: invalid argument (N, nmax, lmax, null pointer or selector)";
        case ETICS_ERR_LIMIT: return "ETICS_ERR_LIMIT: nmax or lmax beyond ETICS_MAX_NMAX / ETICS_MAX_LMAX";
        case ETICS_ERR_ALIGN: return "ETICS_ERR_ALIGN: pointer not 16-byte aligned";
        case ETICS_ERR_WORKSPACE: return "ETICS_ERR_WORKSPACE: workspace too small";
        case ETICS_ERR_CUDA: return "ETICS_ERR_CUDA: CUDA runtime or launch error";
        case ETICS_ERR_STATIC_LIMIT:
            return "ETICS_ERR_STATIC_LIMIT: (nmax+1)(lmax+1)(lmax+2)/2 beyond ETICS_STATIC_MAX_TABLE (1386) of etics_scf_coeffs_static";
        default: return "ETICS: unknown status";
    }
}

etics_status etics_init(void) {
    cudaError_t e = scf_init_constants();
    if (e != cudaSuccess) return ETICS_ERR_CUDA;
    return from_cuda(mex_init_constants());
}

size_t etics_workspace_bytes(int which, long long N, int nmax, int lmax) {
    if (which == ETICS_WS_MEX_FORCE) nmax = 0;
    if (check_sizes(N, nmax, lmax) != ETICS_OK) return 0;
    size_t b = 0;
    switch (which) {
        case ETICS_WS_SCF_COEFFS: b = scf_coeffs_workspace(N, nmax, lmax); break;
        case ETICS_WS_SCF_FORCE: b = 0; break;
        case ETICS_WS_MEX_FORCE: b = mex_workspace(N, lmax); break;
        case ETICS_WS_SCF_FORCE_F32: b = scf_force_f32_workspace(nmax, lmax); break;
        default: return 0;
    }
    return b < 256 ? 256 : round_up(b, 256);
}

etics_status etics_scf_coeffs(const double* pos, const double* mass, long long N, int nmax, int lmax,
                              double* A, double* B, void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, nmax, lmax);
    if (s != ETICS_OK) return s;
    if (!pos || !mass || !A || !B || !workspace) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(mass) || misaligned(A) || misaligned(B) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_SCF_COEFFS, N, nmax, lmax)) return ETICS_ERR_WORKSPACE;
    return from_cuda(scf_coeffs_launch(pos, mass, N, nmax, lmax, A, B, workspace, static_cast<cudaStream_t>(stream)));
}

etics_status etics_scf_force_ex(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                                int what, double* acc, double* pot, void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, nmax, lmax);
    if (s != ETICS_OK) return s;
    (void)workspace; (void)workspace_bytes;   // this call needs no workspace; NULL / 0 are accepted
    if (what != ETICS_WHAT_BOTH && what != ETICS_WHAT_POTENTIAL && what != ETICS_WHAT_FORCE) return ETICS_ERR_ARG;
    if (what == ETICS_WHAT_POTENTIAL) acc = nullptr;
    if (what == ETICS_WHAT_FORCE) pot = nullptr;
    if (!pos || !A || !B || (!acc && what != ETICS_WHAT_POTENTIAL) || (!pot && what != ETICS_WHAT_FORCE)) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(A) || misaligned(B) || misaligned(acc) || misaligned(pot)) return ETICS_ERR_ALIGN;
    return from_cuda(scf_force_launch(pos, N, nmax, lmax, A, B, what, acc, pot, static_cast<cudaStream_t>(stream)));
}

etics_status etics_scf_force(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                             double* acc, double* pot, void* workspace, size_t workspace_bytes, void* stream) {
    return etics_scf_force_ex(pos, N, nmax, lmax, A, B, ETICS_WHAT_BOTH, acc, pot, workspace, workspace_bytes, stream);
}

etics_status etics_mex_force_ex(const double* pos, const double* mass, long long N, int lmax,
                                int what, double* acc, double* pot, void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, 0, lmax);
    if (s != ETICS_OK) return s;
    if (what != ETICS_WHAT_BOTH && what != ETICS_WHAT_POTENTIAL && what != ETICS_WHAT_FORCE) return ETICS_ERR_ARG;
    if (what == ETICS_WHAT_POTENTIAL) acc = nullptr;
    if (what == ETICS_WHAT_FORCE) pot = nullptr;
    if (!pos || !mass || !workspace || (!acc && what != ETICS_WHAT_POTENTIAL) || (!pot && what != ETICS_WHAT_FORCE)) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(mass) || misaligned(acc) || misaligned(pot) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax)) return ETICS_ERR_WORKSPACE;
    return from_cuda(mex_force_launch(pos, mass, N, lmax, what, acc, pot, workspace, static_cast<cudaStream_t>(stream)));
}

etics_status etics_mex_force(const double* pos, const double* mass, long long N, int lmax,
                             double* acc, double* pot, void* workspace, size_t workspace_bytes, void* stream) {
    return etics_mex_force_ex(pos, mass, N, lmax, ETICS_WHAT_BOTH, acc, pot, workspace, workspace_bytes, stream);
}

etics_status etics_scf_force_f32(const double* pos, long long N, int nmax, int lmax, const double* A, const double* B,
                                 int what, double* acc, double* pot, void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, nmax, lmax);
    if (s != ETICS_OK) return s;
    if (what != ETICS_WHAT_BOTH && what != ETICS_WHAT_POTENTIAL && what != ETICS_WHAT_FORCE) return ETICS_ERR_ARG;
    if (what == ETICS_WHAT_POTENTIAL) acc = nullptr;
    if (what == ETICS_WHAT_FORCE) pot = nullptr;
    if (!pos || !A || !B || !workspace || (!acc && what != ETICS_WHAT_POTENTIAL) || (!pot && what != ETICS_WHAT_FORCE)) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(A) || misaligned(B) || misaligned(acc) || misaligned(pot) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_SCF_FORCE_F32, N, nmax, lmax)) return ETICS_ERR_WORKSPACE;
    return from_cuda(scf_force_f32_launch(pos, N, nmax, lmax, A, B, acc, pot, workspace, static_cast<cudaStream_t>(stream)));
}

etics_status etics_scf_combine(const double* parts, int nparts, long long len, double* out, void* stream) {
    if (!parts || !out || nparts < 1 || len < 1) return ETICS_ERR_ARG;
    if (misaligned(parts) || misaligned(out)) return ETICS_ERR_ALIGN;
    return from_cuda(scf_combine_launch(parts, nparts, len, out, static_cast<cudaStream_t>(stream)));
}

etics_status etics_mex_sort(const double* pos, long long N, unsigned long long* keys_sorted, unsigned int* perm,
                            void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, 0, 0);
    if (s != ETICS_OK) return s;
    if (!pos || !keys_sorted || !perm || !workspace) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(keys_sorted) || misaligned(perm) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, 0)) return ETICS_ERR_WORKSPACE;
    return from_cuda(mex_sort_launch(pos, N, keys_sorted, perm, workspace, static_cast<cudaStream_t>(stream)));
}

// ---- radius-partitioned MEX --------------------------------------------------------------------------------
int etics_mex_shard_rows(int lmax) {
    return (lmax < 0 || lmax > ETICS_MAX_LMAX) ? 0 : mex_shard_rows(lmax);
}

etics_status etics_mex_shard_moments(const double* pos, const double* mass, long long N, int lmax, double* totals,
                                     void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, 0, lmax);
    if (s != ETICS_OK) return s;
    if (!pos || !mass || !totals || !workspace) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(mass) || misaligned(totals) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax)) return ETICS_ERR_WORKSPACE;
    return from_cuda(mex_shard_moments_launch(pos, mass, N, lmax, totals, workspace, static_cast<cudaStream_t>(stream)));
}

etics_status etics_mex_shard_bases(const double* parts, int nparts, int rank, int lmax, double* base, void* stream) {
    if (lmax < 0 || nparts < 1 || rank < 0 || rank >= nparts || !parts || !base) return ETICS_ERR_ARG;
    if (lmax > ETICS_MAX_LMAX) return ETICS_ERR_LIMIT;
    if (misaligned(parts) || misaligned(base)) return ETICS_ERR_ALIGN;
    return from_cuda(mex_shard_bases_launch(parts, nparts, rank, lmax, base, static_cast<cudaStream_t>(stream)));
}

etics_status etics_mex_shard_force(long long N, int lmax, int what, const double* base, double* acc, double* pot,
                                   void* workspace, size_t workspace_bytes, void* stream) {
    etics_status s = check_sizes(N, 0, lmax);
    if (s != ETICS_OK) return s;
    if (what != ETICS_WHAT_BOTH && what != ETICS_WHAT_POTENTIAL && what != ETICS_WHAT_FORCE) return ETICS_ERR_ARG;
    if (what == ETICS_WHAT_POTENTIAL) acc = nullptr;
    if (what == ETICS_WHAT_FORCE) pot = nullptr;
    if (!base || !workspace || (!acc && what != ETICS_WHAT_POTENTIAL) || (!pot && what != ETICS_WHAT_FORCE)) return ETICS_ERR_ARG;
    if (misaligned(base) || misaligned(acc) || misaligned(pot) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax)) return ETICS_ERR_WORKSPACE;
    return from_cuda(mex_shard_force_launch(N, lmax, what, base, acc, pot, workspace, static_cast<cudaStream_t>(stream)));
}

// ---- host-buffer entry points ------------------------------------------------------------------------------
// Scratch layout: pos[3N] | mass[N] | acc[3N] | pot[N] | A[T] | B[T] | workspace, each 256-byte aligned.
static size_t seg(size_t doubles) { return round_up(doubles * sizeof(double), 256); }

size_t etics_host_scratch_bytes(int method, long long N, int nmax, int lmax) {
    if (method != 0 && method != 1) return 0;
    if (method == 1) nmax = 0;
    if (check_sizes(N, nmax, lmax) != ETICS_OK) return 0;
    const size_t T = (size_t)(nmax + 1) * num_lm(lmax);
    size_t b = seg(3 * (size_t)N) + seg((size_t)N) + seg(3 * (size_t)N) + seg((size_t)N) + 2 * seg(T);
    b += etics_workspace_bytes(method == 0 ? ETICS_WS_SCF_COEFFS : ETICS_WS_MEX_FORCE, N, nmax, lmax);
    return b;
}

etics_status etics_scf_full_host(const double* pos_h, const double* mass_h, long long N, int nmax, int lmax,
                                 double* A_h, double* B_h, double* acc_h, double* pot_h,
                                 void* device_scratch, size_t scratch_bytes, void* stream) {
    etics_status s = check_sizes(N, nmax, lmax);
    if (s != ETICS_OK) return s;
    if (!pos_h || !mass_h || !acc_h || !pot_h || !device_scratch) return ETICS_ERR_ARG;
    if (misaligned(device_scratch)) return ETICS_ERR_ALIGN;
    if (scratch_bytes < etics_host_scratch_bytes(0, N, nmax, lmax)) return ETICS_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t T = (size_t)(nmax + 1) * num_lm(lmax), n = (size_t)N;
    char* p = static_cast<char*>(device_scratch);
    double* d_pos = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_mass = reinterpret_cast<double*>(p); p += seg(n);
    double* d_acc = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_pot = reinterpret_cast<double*>(p); p += seg(n);
    double* d_A = reinterpret_cast<double*>(p); p += seg(T);
    double* d_B = reinterpret_cast<double*>(p); p += seg(T);
    const size_t wsb = etics_workspace_bytes(ETICS_WS_SCF_COEFFS, N, nmax, lmax);
    if (cudaMemcpyAsync(d_pos, pos_h, 3 * n * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return ETICS_ERR_CUDA;
    if (cudaMemcpyAsync(d_mass, mass_h, n * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return ETICS_ERR_CUDA;
    s = etics_scf_coeffs(d_pos, d_mass, N, nmax, lmax, d_A, d_B, p, wsb, stream);
    if (s != ETICS_OK) return s;
    s = etics_scf_force(d_pos, N, nmax, lmax, d_A, d_B, d_acc, d_pot, nullptr, 0, stream);
    if (s != ETICS_OK) return s;
    if (cudaMemcpyAsync(acc_h, d_acc, 3 * n * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ETICS_ERR_CUDA;
    if (cudaMemcpyAsync(pot_h, d_pot, n * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ETICS_ERR_CUDA;
    if (A_h && cudaMemcpyAsync(A_h, d_A, T * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ETICS_ERR_CUDA;
    if (B_h && cudaMemcpyAsync(B_h, d_B, T * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ETICS_ERR_CUDA;
    return ETICS_OK;
}

etics_status etics_mex_full_host(const double* pos_h, const double* mass_h, long long N, int lmax,
                                 double* acc_h, double* pot_h, void* device_scratch, size_t scratch_bytes, void* stream) {
    etics_status s = check_sizes(N, 0, lmax);
    if (s != ETICS_OK) return s;
    if (!pos_h || !mass_h || !acc_h || !pot_h || !device_scratch) return ETICS_ERR_ARG;
    if (misaligned(device_scratch)) return ETICS_ERR_ALIGN;
    if (scratch_bytes < etics_host_scratch_bytes(1, N, 0, lmax)) return ETICS_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t T = (size_t)num_lm(lmax), n = (size_t)N;
    char* p = static_cast<char*>(device_scratch);
    double* d_pos = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_mass = reinterpret_cast<double*>(p); p += seg(n);
    double* d_acc = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_pot = reinterpret_cast<double*>(p); p += seg(n);
    p += 2 * seg(T);
    const size_t wsb = etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax);
    if (cudaMemcpyAsync(d_pos, pos_h, 3 * n * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return ETICS_ERR_CUDA;
    if (cudaMemcpyAsync(d_mass, mass_h, n * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return ETICS_ERR_CUDA;
    s = etics_mex_force(d_pos, d_mass, N, lmax, d_acc, d_pot, p, wsb, stream);
    if (s != ETICS_OK) return s;
    if (cudaMemcpyAsync(acc_h, d_acc, 3 * n * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ETICS_ERR_CUDA;
    if (cudaMemcpyAsync(pot_h, d_pot, n * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ETICS_ERR_CUDA;
    return ETICS_OK;
}

// ---- one upload, both methods, overlapped copies ------------------------------------------------------------------------
// Scratch layout: pos[3N] | mass[N] | acc_scf[3N] | pot_scf[N] | acc_mex[3N] | pot_mex[N] | A[T] | B[T] | ws_scf | ws_mex.
size_t etics_step_host_scratch_bytes(long long N, int nmax, int lmax, int mex_lmax) {
    if (check_sizes(N, nmax, lmax) != ETICS_OK || check_sizes(N, 0, mex_lmax) != ETICS_OK) return 0;
    const size_t T = (size_t)(nmax + 1) * num_lm(lmax);
    return 2 * (seg(3 * (size_t)N) + seg((size_t)N)) + seg(3 * (size_t)N) + seg((size_t)N) + 2 * seg(T) +
           etics_workspace_bytes(ETICS_WS_SCF_COEFFS, N, nmax, lmax) + etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, mex_lmax);
}

etics_status etics_step_host(const double* pos_h, const double* mass_h, long long N, int nmax, int lmax, int mex_lmax,
                             double* A_h, double* B_h, double* acc_scf_h, double* pot_scf_h, double* acc_mex_h, double* pot_mex_h,
                             void* device_scratch, size_t scratch_bytes, void* stream, void* copy_stream) {
    etics_status s = check_sizes(N, nmax, lmax);
    if (s != ETICS_OK) return s;
    s = check_sizes(N, 0, mex_lmax);
    if (s != ETICS_OK) return s;
    if (!pos_h || !mass_h || !acc_scf_h || !pot_scf_h || !acc_mex_h || !pot_mex_h || !device_scratch) return ETICS_ERR_ARG;
    if (misaligned(device_scratch)) return ETICS_ERR_ALIGN;
    if (scratch_bytes < etics_step_host_scratch_bytes(N, nmax, lmax, mex_lmax)) return ETICS_ERR_WORKSPACE;
    if (etics_init() != ETICS_OK) return ETICS_ERR_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaStream_t cs = copy_stream ? static_cast<cudaStream_t>(copy_stream) : st;
    const bool two = cs != st;
    const size_t T = (size_t)(nmax + 1) * num_lm(lmax), n = (size_t)N;
    char* p = static_cast<char*>(device_scratch);
    double* d_pos = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_mass = reinterpret_cast<double*>(p); p += seg(n);
    double* d_acc1 = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_pot1 = reinterpret_cast<double*>(p); p += seg(n);
    double* d_acc2 = reinterpret_cast<double*>(p); p += seg(3 * n);
    double* d_pot2 = reinterpret_cast<double*>(p); p += seg(n);
    double* d_A = reinterpret_cast<double*>(p); p += seg(T);
    double* d_B = reinterpret_cast<double*>(p); p += seg(T);
    void* ws_scf = p; p += etics_workspace_bytes(ETICS_WS_SCF_COEFFS, N, nmax, lmax);
    void* ws_mex = p;
    const size_t ws_mex_bytes = etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, mex_lmax);

    // events order the two streams; they are destroyed right after the enqueue (CUDA releases them once they have completed)
    constexpr int kMaxChunks = 8;
    cudaEvent_t ev[kMaxChunks + 4] = {};
    int nev = 0;
    bool ok = true;
    auto fail = [&]() { ok = false; };
    auto link = [&](cudaStream_t from, cudaStream_t to) {   // `to` continues after everything enqueued so far on `from`
        if (!two || !ok) return;
        cudaEvent_t e = nullptr;
        if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return fail();
        ev[nev++] = e;
        if (cudaEventRecord(e, from) != cudaSuccess || cudaStreamWaitEvent(to, e, 0) != cudaSuccess) fail();
    };
    auto copy = [&](void* dst, const void* src, size_t bytes, cudaMemcpyKind kind) {
        if (ok && bytes && cudaMemcpyAsync(dst, src, bytes, kind, cs) != cudaSuccess) fail();
    };
    link(st, cs);   // the copies start after the work already on the caller's stream

    // H2D in ranges of whole accumulation blocks; each range is accumulated as soon as it has arrived (coefficients
    // are additive over particles), so the upload hides the coefficient pass
    long long per_block = 0;
    const int blocks = scf_coeffs_blocks(N, nmax, lmax, &per_block);
    const int chunks = !two ? 1 : (blocks < kMaxChunks ? blocks : kMaxChunks);
    for (int c = 0; c < chunks && ok; ++c) {
        const int b0 = (int)((long long)blocks * c / chunks), b1 = (int)((long long)blocks * (c + 1) / chunks);
        const size_t k0 = (size_t)b0 * per_block;
        size_t k1 = (size_t)b1 * per_block;
        if (k1 > n || c == chunks - 1) k1 = n;
        for (int d = 0; d < 3; ++d) copy(d_pos + d * n + k0, pos_h + d * n + k0, (k1 - k0) * 8, cudaMemcpyHostToDevice);
        copy(d_mass + k0, mass_h + k0, (k1 - k0) * 8, cudaMemcpyHostToDevice);
        link(cs, st);
        if (ok && scf_accumulate_launch(d_pos, d_mass, N, nmax, lmax, ws_scf, b0, b1 - b0, st) != cudaSuccess) fail();
    }
    if (ok && scf_finalize_launch(N, nmax, lmax, d_A, d_B, ws_scf, st) != cudaSuccess) fail();
    if (ok && scf_force_launch(d_pos, N, nmax, lmax, d_A, d_B, ETICS_WHAT_BOTH, d_acc1, d_pot1, st) != cudaSuccess) fail();
    link(st, cs);   // the SCF results go home while the MEX kernels run
    copy(acc_scf_h, d_acc1, 3 * n * 8, cudaMemcpyDeviceToHost);
    copy(pot_scf_h, d_pot1, n * 8, cudaMemcpyDeviceToHost);
    if (A_h) copy(A_h, d_A, T * 8, cudaMemcpyDeviceToHost);
    if (B_h) copy(B_h, d_B, T * 8, cudaMemcpyDeviceToHost);
    if (ok && mex_force_launch(d_pos, d_mass, N, mex_lmax, ETICS_WHAT_BOTH, d_acc2, d_pot2, ws_mex, st) != cudaSuccess) fail();
    (void)ws_mex_bytes;
    link(st, cs);
    copy(acc_mex_h, d_acc2, 3 * n * 8, cudaMemcpyDeviceToHost);
    copy(pot_mex_h, d_pot2, n * 8, cudaMemcpyDeviceToHost);
    link(cs, st);   // the caller's stream ends after the last copy
    for (int i = 0; i < nev; ++i) cudaEventDestroy(ev[i]);
    return ok ? ETICS_OK : ETICS_ERR_CUDA;
}

// ---- measurement support ---------------------------------------------------------------------------------
etics_status etics_mex_force_timed(const double* pos, const double* mass, long long N, int lmax,
                                   double* acc, double* pot, void* workspace, size_t workspace_bytes, void* stream,
                                   float* stage_ms) {
    etics_status s = check_sizes(N, 0, lmax);
    if (s != ETICS_OK) return s;
    if (!pos || !mass || !acc || !pot || !workspace || !stage_ms) return ETICS_ERR_ARG;
    if (misaligned(pos) || misaligned(mass) || misaligned(acc) || misaligned(pot) || misaligned(workspace)) return ETICS_ERR_ALIGN;
    if (workspace_bytes < etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax)) return ETICS_ERR_WORKSPACE;
    return from_cuda(mex_force_timed(pos, mass, N, lmax, acc, pot, workspace, static_cast<cudaStream_t>(stream), stage_ms));
}

int etics_kernel_launches(int which, long long N) {
    switch (which) {
        case ETICS_WS_SCF_COEFFS: return 2;
        case ETICS_WS_SCF_FORCE: return 1;
        case ETICS_WS_MEX_FORCE: return (N >= 1 && N < (1LL << 31)) ? mex_kernel_launches(N) : 0;
        default: return 0;
    }
}

// ---- probes ----------------------------------------------------------------------------------------------
etics_status etics_probe_dfma(int iters, double* sink, double* flops_out, void* stream) {
    if (iters < 1 || !sink) return ETICS_ERR_ARG;
    return from_cuda(probe_dfma_launch(iters, sink, flops_out, static_cast<cudaStream_t>(stream)));
}

etics_status etics_probe_copy(void* dst, const void* src, size_t bytes, void* stream) {
    if (!dst || !src || bytes < 16) return ETICS_ERR_ARG;
    if (misaligned(dst) || misaligned(src)) return ETICS_ERR_ALIGN;
    return from_cuda(probe_copy_launch(dst, src, bytes, static_cast<cudaStream_t>(stream)));
}

}  // extern "C"

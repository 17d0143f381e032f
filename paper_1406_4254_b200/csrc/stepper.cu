// stepper.cu — time-stepping reuse of the force path: the paper evolves its systems with a leapfrog
// that calls the force routine once per step (§3.4: "after the system is evolved one very short leapfrog
// time step").  A stepper owns NO device memory: it refers to the caller's pos / vel / mass / acc / pot and workspace,
// keeps the launch sequence of one kick-drift-kick step as a CUDA graph (optional) and replays it.
//
//   step:  v += (dt/2) a(x);  x += dt v;  a = force(x);  v += (dt/2) a(x)        (kick-drift-kick, eq. of motion x'' = a)
//
// The first half kick and the drift are one kernel, the closing half kick another; the force in between is the
// unchanged launch sequence of etics_scf_coeffs + etics_scf_force, or of etics_mex_force (from the UNSORTED list: an LSD
// radix sort does the same work whether or not the list is nearly sorted).
#include <new>

#include "etics_common.cuh"

namespace etics {

__global__ void __launch_bounds__(256)
leapfrog_kick_drift_kernel(double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ acc, long long n3,
                           double half_dt, double dt) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    const double v = fma(half_dt, acc[i], vel[i]);
    vel[i] = v;
    pos[i] = fma(dt, v, pos[i]);
}

__global__ void __launch_bounds__(256)
leapfrog_kick_kernel(double* __restrict__ vel, const double* __restrict__ acc, long long n3, double half_dt) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    vel[i] = fma(half_dt, acc[i], vel[i]);
}

}  // namespace etics

using namespace etics;

struct etics_stepper {
    int method, nmax, lmax, use_graph;
    long long N;
    double dt;
    double *pos, *vel, *acc, *pot;
    const double* mass;
    double *A, *B;          // SCF: inside the workspace
    void* ws;               // force workspace
    size_t ws_bytes;
    cudaStream_t stream;
    cudaGraph_t graph[2];       // [0] step with fresh coefficients, [1] step with the held coefficients (SCF only)
    cudaGraphExec_t exec[2];
    bool have_acc;          // acc holds a(pos)
    int every;              // SCF: coefficients are recomputed at force evaluations 0, every, 2 every, ... (temporal softening)
    long long evals;        // force evaluations so far
};

namespace {

size_t stepper_table_bytes(int nmax, int lmax) { return round_up((size_t)(nmax + 1) * num_lm(lmax) * sizeof(double), 256); }

etics_status stepper_force(etics_stepper* s, bool fresh) {
    if (s->method == 0) {
        if (fresh) {
            const etics_status e = etics_scf_coeffs(s->pos, s->mass, s->N, s->nmax, s->lmax, s->A, s->B, s->ws, s->ws_bytes, s->stream);
            if (e != ETICS_OK) return e;
        }
        return etics_scf_force(s->pos, s->N, s->nmax, s->lmax, s->A, s->B, s->acc, s->pot, nullptr, 0, s->stream);
    }
    return etics_mex_force(s->pos, s->mass, s->N, s->lmax, s->acc, s->pot, s->ws, s->ws_bytes, s->stream);
}

etics_status stepper_enqueue_step(etics_stepper* s, bool fresh) {
    const long long n3 = 3 * s->N;
    const unsigned blocks = (unsigned)((n3 + 255) / 256);
    leapfrog_kick_drift_kernel<<<blocks, 256, 0, s->stream>>>(s->pos, s->vel, s->acc, n3, 0.5 * s->dt, s->dt);
    if (cudaGetLastError() != cudaSuccess) return ETICS_ERR_CUDA;
    etics_status e = stepper_force(s, fresh);
    if (e != ETICS_OK) return e;
    leapfrog_kick_kernel<<<blocks, 256, 0, s->stream>>>(s->vel, s->acc, n3, 0.5 * s->dt);
    return cudaGetLastError() == cudaSuccess ? ETICS_OK : ETICS_ERR_CUDA;
}

}  // namespace

extern "C" {

size_t etics_stepper_workspace_bytes(int method, long long N, int nmax, int lmax) {
    if (method == 0) {
        const size_t w = etics_workspace_bytes(ETICS_WS_SCF_COEFFS, N, nmax, lmax);
        return w ? w + 2 * stepper_table_bytes(nmax, lmax) : 0;
    }
    if (method == 1) return etics_workspace_bytes(ETICS_WS_MEX_FORCE, N, 0, lmax);
    return 0;
}

etics_status etics_stepper_create(etics_stepper** out, int method, double* pos, double* vel, const double* mass, long long N,
                                  int nmax, int lmax, double dt, double* acc, double* pot,
                                  void* workspace, size_t workspace_bytes, int use_graph, void* stream) {
    if (!out) return ETICS_ERR_ARG;
    *out = nullptr;
    if (method != 0 && method != 1) return ETICS_ERR_ARG;
    if (method == 1) nmax = 0;
    const size_t need = etics_stepper_workspace_bytes(method, N, nmax, lmax);
    if (need == 0) return (N < 1 || N >= (1LL << 31) || nmax < 0 || lmax < 0) ? ETICS_ERR_ARG : ETICS_ERR_LIMIT;
    if (!pos || !vel || !mass || !acc || !pot || !workspace) return ETICS_ERR_ARG;
    for (const void* p : {(const void*)pos, (const void*)vel, (const void*)mass, (const void*)acc, (const void*)pot, (const void*)workspace})
        if (reinterpret_cast<uintptr_t>(p) & 15u) return ETICS_ERR_ALIGN;
    if (workspace_bytes < need) return ETICS_ERR_WORKSPACE;
    etics_status st = etics_init();   // per-device set-up must not happen inside a stream capture
    if (st != ETICS_OK) return st;
    etics_stepper* s = new (std::nothrow) etics_stepper{};
    if (!s) return ETICS_ERR_CUDA;
    s->method = method; s->nmax = nmax; s->lmax = lmax; s->use_graph = use_graph; s->N = N; s->dt = dt;
    s->pos = pos; s->vel = vel; s->mass = mass; s->acc = acc; s->pot = pot;
    s->stream = static_cast<cudaStream_t>(stream);
    char* w = static_cast<char*>(workspace);
    if (method == 0) {
        s->A = reinterpret_cast<double*>(w); w += stepper_table_bytes(nmax, lmax);
        s->B = reinterpret_cast<double*>(w); w += stepper_table_bytes(nmax, lmax);
        s->ws_bytes = workspace_bytes - 2 * stepper_table_bytes(nmax, lmax);
    } else {
        s->ws_bytes = workspace_bytes;
    }
    s->ws = w;
    s->every = 1;
    if (use_graph) {
        // the step's launch sequence is recorded once; replaying it costs one launch per step instead of 4-17.  It is
        // recorded on a stream of its own (capturing work is not executed, and the caller's stream may be the legacy
        // default stream, which cannot capture); the graph is then launched on the caller's stream.
        cudaStream_t cap = nullptr, user = s->stream;
        if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) != cudaSuccess) { delete s; return ETICS_ERR_CUDA; }
        etics_status e = ETICS_OK;
        for (int v = 0; v < (method == 0 ? 2 : 1) && e == ETICS_OK; ++v) {
            e = ETICS_ERR_CUDA;
            cudaGraph_t g = nullptr;
            if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                s->stream = cap;
                e = stepper_enqueue_step(s, v == 0);
                s->stream = user;
                if (cudaStreamEndCapture(cap, &g) != cudaSuccess && e == ETICS_OK) e = ETICS_ERR_CUDA;
            }
            s->graph[v] = g;
            if (e == ETICS_OK && (!g || cudaGraphInstantiate(&s->exec[v], g, 0) != cudaSuccess)) e = ETICS_ERR_CUDA;
        }
        cudaStreamDestroy(cap);
        if (e != ETICS_OK) {
            for (int v = 0; v < 2; ++v) { if (s->exec[v]) cudaGraphExecDestroy(s->exec[v]); if (s->graph[v]) cudaGraphDestroy(s->graph[v]); }
            delete s;
            cudaGetLastError();
            return e;
        }
    }
    *out = s;
    return ETICS_OK;
}

etics_status etics_stepper_set_coefficient_interval(etics_stepper* s, int every) {
    if (!s || every < 1 || s->method != 0 || s->have_acc) return ETICS_ERR_ARG;
    s->every = every;
    return ETICS_OK;
}

etics_status etics_stepper_step(etics_stepper* s, int nsteps) {
    if (!s || nsteps < 0) return ETICS_ERR_ARG;
    if (!s->have_acc) {   // a(x_0): force evaluation 0
        const etics_status e = stepper_force(s, true);
        if (e != ETICS_OK) return e;
        s->have_acc = true;
        s->evals = 1;
    }
    for (int i = 0; i < nsteps; ++i, ++s->evals) {
        const bool fresh = s->method != 0 || s->evals % s->every == 0;
        cudaGraphExec_t g = s->exec[fresh ? 0 : 1];
        if (g) {
            if (cudaGraphLaunch(g, s->stream) != cudaSuccess) return ETICS_ERR_CUDA;
        } else {
            const etics_status e = stepper_enqueue_step(s, fresh);
            if (e != ETICS_OK) return e;
        }
    }
    return ETICS_OK;
}

etics_status etics_stepper_destroy(etics_stepper* s) {
    if (!s) return ETICS_OK;
    cudaError_t e = cudaSuccess;
    if (s->exec[0]) e = cudaStreamSynchronize(s->stream);   // a graph must not be in flight when it is destroyed
    for (int v = 0; v < 2; ++v) {
        if (s->exec[v]) cudaGraphExecDestroy(s->exec[v]);
        if (s->graph[v]) cudaGraphDestroy(s->graph[v]);
    }
    delete s;
    return e == cudaSuccess ? ETICS_OK : ETICS_ERR_CUDA;
}

}  // extern "C"

// ea_api.cu -- the C ABI of libea_b200.so (declared in include/ea.h): argument checking, device memory,
// launch sequencing.  No arithmetic of the method lives here except the acceptance thresholds (Eq. 9).
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <exception>
#include <new>

#include "ea_internal.h"

namespace ea {

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

WorkspaceLayout workspace_layout(int L, int n_samples, int n_replicas, int n_slots)
{
    WorkspaceLayout w;
    size_t N = (size_t)L * L * L, bond_bytes = n_replicas == 2 ? 4 : 8;
    w.n_counters = (size_t)(3 * (L / 2 + 1) + 1) * 64;
    size_t off = 0;
    w.off_spins = off;    off = align_up(off + N * 8);
    w.off_bonds = off;    off = align_up(off + 3 * N * bond_bytes);
    w.off_snaps = off;    off = align_up(off + (size_t)n_slots * N * 8);
    w.off_stage = off;    off = align_up(off + N * 8);
    w.off_counters = off; off = align_up(off + w.n_counters * 8);
    w.off_time = off;     off = align_up(off + 8);
    w.off_flags = off;    off = align_up(off + resident_aux_bytes());
    w.off_fold = off;     off = align_up(off + fold_bytes(L, n_samples));
    w.total = off;
    return w;
}

static int ilog2_exact(unsigned v)
{
    if (v == 0 || (v & (v - 1))) return -1;
    int l = 0;
    while ((1u << l) != v) ++l;
    return l;
}

// Eq. 9 with sum_j J_ij S_i S_j = 6 - 2 n_u:  thr[n_u] = floor(2^32 exp(-4 (3 - n_u) / T) + 0.5),
// n_u = 0, 1, 2 (C-A4).  T = 0 -> exp(-inf) = 0;  T = +inf -> exp(-0) = 1 -> 2^32 ("always").
static void compute_thresholds(double T, uint64_t thr[3], Thresholds &th)
{
    for (int k = 0; k < 3; ++k) {
        double w = exp(-(4.0 * (double)(3 - k)) / T);
        thr[k] = (uint64_t)floor(4294967296.0 * w + 0.5);
        th.thr[k] = thr[k] > 0xffffffffull ? 0xffffffffu : (uint32_t)thr[k];
        th.always[k] = thr[k] > 0xffffffffull ? 0xffffffffu : 0u;
    }
}

// Heat bath (C-HB): thr[n_u] = floor(2^32 / (1 + exp((12 - 4 n_u) / T)) + 0.5); Delta E = 0 is exactly 1/2 at any T.
static void compute_thresholds_heatbath(double T, uint64_t thr[7], Thresholds &th)
{
    for (int k = 0; k < 7; ++k) {
        const double dE = 12.0 - 4.0 * (double)k;
        const double w = dE == 0.0 ? 1.0 : exp(dE / T);
        thr[k] = (uint64_t)floor(4294967296.0 * (1.0 / (1.0 + w)) + 0.5);
        th.hb[k] = thr[k] > 0xffffffffull ? 0xffffffffu : (uint32_t)thr[k];
        th.hb_always[k] = thr[k] > 0xffffffffull ? 0xffffffffu : 0u;
    }
}

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
        changed = ok && prev != dev;
    }
    ~DeviceGuard() { if (changed) cudaSetDevice(prev); }
    bool changed = false;
};

} // namespace ea

using namespace ea;

#define EA_FAIL(sim, code, ...)                                   \
    do {                                                          \
        char _b[512];                                             \
        snprintf(_b, sizeof(_b), __VA_ARGS__);                    \
        if (sim) (sim)->err = _b;                                 \
        return (code);                                            \
    } while (0)

#define EA_CUDA(sim, expr)                                                                     \
    do {                                                                                       \
        cudaError_t _e = (expr);                                                               \
        if (_e != cudaSuccess) EA_FAIL(sim, EA_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(_e)); \
    } while (0)

// Wait for the sim's stream; if a RESIDENT launch ran since the last check, read its abort word (a CTA whose
// neighbour never published its step gives up after 2 s instead of hanging the device).
static ea_status stream_sync(ea_sim *s)
{
    EA_CUDA(s, cudaStreamSynchronize(s->stream));
    if (s->resident_used) {
        s->resident_used = false;
        unsigned *d_abort = s->resident_flags + (resident_flag_bytes() / sizeof(unsigned) - 32);
        unsigned aborted = 0;
        EA_CUDA(s, cudaMemcpy(&aborted, d_abort, sizeof(aborted), cudaMemcpyDeviceToHost));
        if (aborted) {
            cudaMemset(s->resident_flags, 0, resident_flag_bytes());
            s->resident_epoch = 0;
            EA_FAIL(s, EA_ERR_CUDA, "resident sweep kernel: neighbour wait timed out; the spin state is invalid");
        }
    }
    return EA_OK;
}
#define EA_SYNC(sim)                          \
    do {                                      \
        ea_status _rc = stream_sync(sim);     \
        if (_rc != EA_OK) return _rc;         \
    } while (0)

static const uint64_t RESIDENT_AUTO_MIN_SWEEPS = 8;     // AUTO: below this the prologue/epilogue of the persistent kernel does not pay
static const uint64_t SMALL_AUTO_MIN_SWEEPS = 2;         // AUTO: a single sweep is two direct launches
static const uint64_t PERSISTENT_MIN_SWEEPS = 4;         // ROWS_PERSISTENT: below this the per-colour launches are as good
static const uint64_t RESIDENT_MAX_SWEEPS = 1u << 20;   // sweeps per persistent launch (about 10 s of device time)

static bool valid_L(int L) { return L >= 2 && (L & 1) == 0 && (int64_t)L * L * L < ((int64_t)1 << 31); }

static bool kernel_valid_for(int kernel, int L)
{
    switch (kernel) {
    case EA_KERNEL_SCALAR: return true;
    case EA_KERNEL_VEC2: return L % 4 == 0;
    case EA_KERNEL_ROWS: return L == 16 || L == 32 || L == 64 || L == 128;
    case EA_KERNEL_RESIDENT: return L == 128; // plus a device check (resident_supported) once the sim exists
    case EA_KERNEL_ROWS_PERSISTENT: return rows_persistent_valid(L);
    case EA_KERNEL_SMALL: return small_cluster_size(L, 1) > 0; // plus a device check (small_supported)
    case EA_KERNEL_FOLD: return false;        // not selectable: it is what a sim with n_samples < 64 runs
    default: return false;
    }
}

static int resolve_kernel(int kernel, int L)
{
    if (kernel == EA_KERNEL_AUTO)
        return kernel_valid_for(EA_KERNEL_ROWS, L) ? EA_KERNEL_ROWS : L % 4 == 0 ? EA_KERNEL_VEC2 : EA_KERNEL_SCALAR;
    return kernel;
}

extern "C" {

const char *ea_version(void) { return "ea_b200 0.1 (sm_100a)"; }

const char *ea_strerror(ea_status s)
{
    switch (s) {
    case EA_OK: return "ok";
    case EA_ERR_INVALID: return "invalid argument";
    case EA_ERR_CUDA: return "CUDA error";
    case EA_ERR_NOMEM: return "out of memory";
    case EA_ERR_STATE: return "invalid state";
    }
    return "unknown status";
}

const char *ea_last_error(const ea_sim *sim) { return sim ? sim->err.c_str() : "null handle"; }

size_t ea_workspace_bytes(int L, int n_replicas, int n_slots) { return ea_workspace_bytes_ex(L, EA_LANES, n_replicas, n_slots); }

size_t ea_workspace_bytes_ex(int L, int n_samples, int n_replicas, int n_slots)
{
    if (!valid_L(L) || (n_replicas != 1 && n_replicas != 2) || n_slots < 0 || !fold_valid(L, n_samples, n_replicas)) return 0;
    return workspace_layout(L, n_samples, n_replicas, n_slots).total;
}

static void destroy_graph(ea_sim *s)
{
    if (s->graph_exec) cudaGraphExecDestroy(s->graph_exec);
    s->graph_exec = nullptr;
    s->graph_sweeps = 0;
}

ea_status ea_destroy(ea_sim *sim)
{
    if (!sim) return EA_OK;
    {
        DeviceGuard g(sim->device);
        cudaStreamSynchronize(sim->stream);
        destroy_graph(sim);
        if (sim->c4v_jobs) cudaFree(sim->c4v_jobs);
        if (sim->c4v_out) cudaFree(sim->c4v_out);
        if (sim->own_ws && sim->ws) cudaFree(sim->ws);
        if (sim->own_stream && sim->stream) cudaStreamDestroy(sim->stream);
    }
    delete sim;
    return EA_OK;
}

ea_status ea_create_ex(const ea_params *prm, ea_sim **out)
{
    if (!prm || !out) return EA_ERR_INVALID;
    if (!valid_L(prm->L) || (prm->n_replicas != 1 && prm->n_replicas != 2) ||
        !fold_valid(prm->L, prm->n_samples, prm->n_replicas) ||
        prm->n_slots < 0 || !(prm->p >= 0.0 && prm->p <= 1.0) || !(prm->T >= 0.0))
        return EA_ERR_INVALID;
    int kernel = resolve_kernel(prm->kernel, prm->L);
    if (!kernel_valid_for(kernel, prm->L)) return EA_ERR_INVALID;

    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) return EA_ERR_CUDA; // no CPU fallback
    int device = prm->device;
    if (device < 0 && cudaGetDevice(&device) != cudaSuccess) return EA_ERR_CUDA;
    if (device >= n_dev) return EA_ERR_INVALID;

    ea_sim *s = new (std::nothrow) ea_sim();
    if (!s) return EA_ERR_NOMEM;
    const int L = prm->L;
    s->lat.L = L;
    s->lat.Lh = L / 2;
    s->lat.log2L = ilog2_exact(L);
    s->lat.log2Lh = ilog2_exact(L / 2);
    s->N = (int64_t)L * L * L;
    s->lat.Nh = (unsigned)(s->N / 2);
    s->n_replicas = prm->n_replicas;
    s->n_samples = prm->n_samples;
    s->n_slots = prm->n_slots;
    s->p = prm->p;
    s->T = prm->T;
    s->seed = prm->seed;
    s->t = 0;
    s->device = device;
    s->kernel = kernel;
    compute_thresholds(s->T, s->thr, s->th);
    compute_thresholds_heatbath(s->T, s->thr_hb, s->th);
    s->slot_set.assign(prm->n_slots, 0);
    s->slot_t.assign(prm->n_slots, 0);

    DeviceGuard g(device);
    ea_status rc = EA_OK;
    cudaError_t e = cudaSuccess;
    WorkspaceLayout w = workspace_layout(L, s->n_samples, s->n_replicas, s->n_slots);
    do {
        if (!g.ok) { rc = EA_ERR_CUDA; break; }
        cudaDeviceGetAttribute(&s->n_sm, cudaDevAttrMultiProcessorCount, device);
        if (prm->stream) {
            if ((cudaStream_t)prm->stream == cudaStreamLegacy) { // cannot be captured into a graph (ea_sweep would fail late)
                fprintf(stderr, "ea_create_ex: the legacy default stream is not supported; pass NULL or a created stream\n");
                rc = EA_ERR_INVALID;
                break;
            }
            s->stream = (cudaStream_t)prm->stream;
        } else { // own stream: the legacy default stream cannot be captured into a graph
            if ((e = cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
            s->own_stream = true;
        }
        if (prm->d_workspace) {
            if (prm->workspace_bytes < w.total || ((uintptr_t)prm->d_workspace & 255)) { rc = EA_ERR_NOMEM; break; }
            s->ws = (char *)prm->d_workspace;
        } else {
            if ((e = cudaMalloc((void **)&s->ws, w.total)) != cudaSuccess) { rc = EA_ERR_NOMEM; break; }
            s->own_ws = true;
        }
        s->ws_bytes = w.total;
        s->spins = (uint64_t *)(s->ws + w.off_spins);
        s->bonds = (void *)(s->ws + w.off_bonds);
        s->snaps = (uint64_t *)(s->ws + w.off_snaps);
        s->stage = (uint64_t *)(s->ws + w.off_stage);
        s->counters = (unsigned long long *)(s->ws + w.off_counters);
        s->n_counters = w.n_counters;
        s->d_time = (uint64_t *)(s->ws + w.off_time);
        s->resident_flags = (unsigned *)(s->ws + w.off_flags);
        if ((e = cudaMemsetAsync(s->resident_flags, 0, resident_flag_bytes(), s->stream)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
        if (const char *ms = getenv("EA_RESIDENT_TIMEOUT_MS")) {
            const long long v = atoll(ms);
            if (v > 0) s->resident_timeout_ns = (uint64_t)v * 1000000ull;
        }
        std::string why;
        if (kernel_valid_for(EA_KERNEL_RESIDENT, L) && resident_supported(s, &why) && (e = resident_prepare(s, &why)) != cudaSuccess) {
            fprintf(stderr, "ea_create_ex: %s\n", why.c_str());
            rc = EA_ERR_CUDA;
            break;
        }
        if (prm->kernel == EA_KERNEL_AUTO && kernel_valid_for(EA_KERNEL_RESIDENT, L) && resident_supported(s, &why)) {
            s->kernel = EA_KERNEL_RESIDENT; // long runs in one persistent launch, short ones as ROWS launches
            s->resident_min_sweeps = RESIDENT_AUTO_MIN_SWEEPS;
        } else if (s->kernel == EA_KERNEL_RESIDENT && !resident_supported(s, &why)) {
            fprintf(stderr, "ea_create_ex: %s\n", why.c_str()); // no handle to carry the message yet
            rc = EA_ERR_INVALID;
            break;
        } else if (prm->kernel == EA_KERNEL_AUTO && prm->n_samples == EA_LANES && kernel_valid_for(EA_KERNEL_SMALL, L) && small_supported(s)) {
            s->kernel = EA_KERNEL_SMALL; // calls of two sweeps or more in one launch, lattice in shared memory
            s->resident_min_sweeps = SMALL_AUTO_MIN_SWEEPS;
        } else if (s->kernel == EA_KERNEL_SMALL && !small_supported(s, &why)) {
            fprintf(stderr, "ea_create_ex: %s\n", why.c_str());
            rc = EA_ERR_INVALID;
            break;
        }
        s->h_counters.resize(w.n_counters);
        if ((e = launch_init_bonds(s)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
        if ((e = launch_init_spins(s)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
        if (s->n_samples < EA_LANES) { // mixed multispin coding: the sweeps run on folded words (ea_fold.cu)
            s->f_spins = (uint64_t *)(s->ws + w.off_fold);
            s->f_bonds = s->f_spins + (size_t)2 * (s->lat.Nh / (EA_LANES / s->n_samples));
            s->kernel = EA_KERNEL_FOLD;
            if ((e = fold_from_standard(s, true, true)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
        }
        if ((e = cudaMemsetAsync(s->d_time, 0, 8, s->stream)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
        if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) { rc = EA_ERR_CUDA; break; }
    } while (0);
    if (rc != EA_OK) {
        if (e != cudaSuccess) fprintf(stderr, "ea_create_ex: %s\n", cudaGetErrorString(e));
        if (s->own_ws && s->ws) cudaFree(s->ws);
        if (s->own_stream && s->stream) cudaStreamDestroy(s->stream);
        delete s;
        return rc;
    }
    *out = s;
    return EA_OK;
}

ea_status ea_create(int L, double p, double T, int n_samples, uint64_t seed, ea_sim **out)
{
    ea_params prm;
    memset(&prm, 0, sizeof(prm));
    prm.L = L; prm.n_samples = n_samples; prm.n_replicas = 1; prm.n_slots = 2;
    prm.p = p; prm.T = T; prm.seed = seed; prm.device = -1; prm.kernel = EA_KERNEL_AUTO;
    return ea_create_ex(&prm, out);
}

// ---- dynamics -------------------------------------------------------------------------------------

static const int GRAPH_SWEEPS = 32; // sweeps per CUDA-graph replay (2 kernel nodes each + the time bump)

static ea_status build_graph(ea_sim *s)
{
    destroy_graph(s);
    cudaGraph_t graph = nullptr;
    EA_CUDA(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
    cudaError_t e = cudaSuccess;
    s->capturing = true; // captured nodes are counted per replay, not here
    for (int k = 0; k < GRAPH_SWEEPS && e == cudaSuccess; ++k) {
        e = launch_half_sweep(s, 0, 0, s->d_time, (uint32_t)k, s->stream);
        if (e == cudaSuccess) e = launch_half_sweep(s, 1, 0, s->d_time, (uint32_t)k, s->stream);
    }
    if (e == cudaSuccess) e = launch_bump_time(s, GRAPH_SWEEPS, s->stream);
    cudaError_t e2 = cudaStreamEndCapture(s->stream, &graph);
    s->capturing = false;
    if (e != cudaSuccess || e2 != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        EA_FAIL(s, EA_ERR_CUDA, "graph capture: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
    }
    e = cudaGraphInstantiate(&s->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
        s->graph_exec = nullptr;
        EA_FAIL(s, EA_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
    }
    s->graph_sweeps = GRAPH_SWEEPS;
    s->graph_kernel = s->kernel;
    return EA_OK;
}

ea_status ea_sweep(ea_sim *sim, uint64_t n)
{
    if (!sim) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    uint64_t left = n;
    if (n && sim->n_samples < EA_LANES) sim->unfolded_valid = false; // the standard-layout mirror goes stale
    if (sim->kernel == EA_KERNEL_RESIDENT && n >= sim->resident_min_sweeps) {
        while (left) {
            const uint32_t chunk = (uint32_t)(left < RESIDENT_MAX_SWEEPS ? left : RESIDENT_MAX_SWEEPS);
            EA_CUDA(sim, launch_sweeps_resident(sim, sim->t, chunk, sim->stream));
            sim->resident_used = true;
            sim->t += chunk;
            left -= chunk;
        }
        return EA_OK;
    }
    if (sim->kernel == EA_KERNEL_SMALL && n >= sim->resident_min_sweeps) {
        while (left) {
            const uint32_t chunk = (uint32_t)(left < RESIDENT_MAX_SWEEPS ? left : RESIDENT_MAX_SWEEPS);
            EA_CUDA(sim, launch_sweeps_small(sim, sim->t, chunk, sim->stream));
            sim->t += chunk;
            left -= chunk;
        }
        return EA_OK;
    }
    if (sim->kernel == EA_KERNEL_ROWS_PERSISTENT && sim->dynamics == EA_DYN_METROPOLIS && n >= PERSISTENT_MIN_SWEEPS) {
        while (left) {
            const uint32_t chunk = (uint32_t)(left < RESIDENT_MAX_SWEEPS ? left : RESIDENT_MAX_SWEEPS);
            EA_CUDA(sim, launch_sweeps_rows_persistent(sim, sim->t, chunk, sim->stream));
            sim->t += chunk;
            left -= chunk;
        }
        return EA_OK;
    }
    if (left >= (uint64_t)GRAPH_SWEEPS) {
        if (!sim->graph_exec || sim->graph_kernel != sim->kernel) {
            ea_status rc = build_graph(sim);
            if (rc != EA_OK) return rc;
        }
        // pageable source: staged before the call returns, so &sim->t need not outlive it
        EA_CUDA(sim, cudaMemcpyAsync(sim->d_time, &sim->t, 8, cudaMemcpyHostToDevice, sim->stream));
        while (left >= (uint64_t)sim->graph_sweeps) {
            EA_CUDA(sim, cudaGraphLaunch(sim->graph_exec, sim->stream));
            sim->count_launch(2 * sim->graph_sweeps + 1);
            sim->t += sim->graph_sweeps;
            left -= sim->graph_sweeps;
        }
    }
    for (; left; --left) {
        EA_CUDA(sim, launch_half_sweep(sim, 0, sim->t, nullptr, 0, sim->stream));
        EA_CUDA(sim, launch_half_sweep(sim, 1, sim->t, nullptr, 0, sim->stream));
        sim->t += 1;
    }
    return EA_OK;
}

ea_status ea_half_sweep(ea_sim *sim, int parity)
{
    if (!sim) return EA_ERR_INVALID;
    if (parity != 0 && parity != 1) EA_FAIL(sim, EA_ERR_INVALID, "parity must be 0 or 1");
    DeviceGuard g(sim->device);
    EA_CUDA(sim, launch_half_sweep(sim, parity, sim->t, nullptr, 0, sim->stream));
    if (sim->n_samples < EA_LANES) sim->unfolded_valid = false;
    return EA_OK;
}

ea_status ea_get_time(const ea_sim *sim, uint64_t *t)
{
    if (!sim || !t) return EA_ERR_INVALID;
    *t = sim->t;
    return EA_OK;
}

ea_status ea_set_time(ea_sim *sim, uint64_t t)
{
    if (!sim) return EA_ERR_INVALID;
    sim->t = t;
    return EA_OK;
}

ea_status ea_set_temperature(ea_sim *sim, double T)
{
    if (!sim) return EA_ERR_INVALID;
    if (!(T >= 0.0)) EA_FAIL(sim, EA_ERR_INVALID, "T must be >= 0");
    sim->T = T;
    compute_thresholds(T, sim->thr, sim->th);
    compute_thresholds_heatbath(T, sim->thr_hb, sim->th);
    DeviceGuard g(sim->device);
    destroy_graph(sim); // thresholds are baked into the captured launches
    return EA_OK;
}

ea_status ea_get_thresholds(const ea_sim *sim, uint64_t thr[3])
{
    if (!sim || !thr) return EA_ERR_INVALID;
    memcpy(thr, sim->thr, sizeof(sim->thr));
    return EA_OK;
}

ea_status ea_set_dynamics(ea_sim *sim, int dynamics)
{
    if (!sim) return EA_ERR_INVALID;
    if (dynamics != EA_DYN_METROPOLIS && dynamics != EA_DYN_HEATBATH) EA_FAIL(sim, EA_ERR_INVALID, "unknown dynamics %d", dynamics);
    if (dynamics != sim->dynamics) {
        DeviceGuard g(sim->device);
        destroy_graph(sim); // the captured launches are of the other rule's kernels
        sim->dynamics = dynamics;
    }
    return EA_OK;
}

ea_status ea_get_dynamics(const ea_sim *sim, int *dynamics)
{
    if (!sim || !dynamics) return EA_ERR_INVALID;
    *dynamics = sim->dynamics;
    return EA_OK;
}

ea_status ea_get_thresholds_heatbath(const ea_sim *sim, uint64_t thr[7])
{
    if (!sim || !thr) return EA_ERR_INVALID;
    memcpy(thr, sim->thr_hb, sizeof(sim->thr_hb));
    return EA_OK;
}

ea_status ea_set_concurrency_hint(ea_sim *sim, int n_concurrent_sims)
{
    if (!sim) return EA_ERR_INVALID;
    if (n_concurrent_sims < 1) EA_FAIL(sim, EA_ERR_INVALID, "ea_set_concurrency_hint: n_concurrent_sims %d < 1", n_concurrent_sims);
    sim->n_concurrent = n_concurrent_sims;
    return EA_OK;
}

ea_status ea_set_kernel(ea_sim *sim, int kernel)
{
    if (!sim) return EA_ERR_INVALID;
    if (sim->n_samples < EA_LANES) {
        if (kernel == EA_KERNEL_AUTO || kernel == EA_KERNEL_FOLD) return EA_OK;
        EA_FAIL(sim, EA_ERR_STATE, "a sim with n_samples < 64 runs the folded kernel only");
    }
    int k = resolve_kernel(kernel, sim->lat.L);
    if (!kernel_valid_for(k, sim->lat.L)) EA_FAIL(sim, EA_ERR_INVALID, "kernel %d not valid for L=%d", kernel, sim->lat.L);
    sim->resident_min_sweeps = 1;
    if (kernel == EA_KERNEL_AUTO && kernel_valid_for(EA_KERNEL_RESIDENT, sim->lat.L) && resident_supported(sim)) {
        k = EA_KERNEL_RESIDENT;
        sim->resident_min_sweeps = RESIDENT_AUTO_MIN_SWEEPS;
    }
    else if (kernel == EA_KERNEL_AUTO && kernel_valid_for(EA_KERNEL_SMALL, sim->lat.L) && small_supported(sim)) {
        k = EA_KERNEL_SMALL;
        sim->resident_min_sweeps = SMALL_AUTO_MIN_SWEEPS;
    }
    std::string why;
    if (k == EA_KERNEL_RESIDENT && !resident_supported(sim, &why)) EA_FAIL(sim, EA_ERR_INVALID, "%s", why.c_str());
    if (k == EA_KERNEL_SMALL && !small_supported(sim, &why)) EA_FAIL(sim, EA_ERR_INVALID, "%s", why.c_str());
    sim->kernel = k;
    return EA_OK;
}

ea_status ea_get_kernel(const ea_sim *sim, int *kernel)
{
    if (!sim || !kernel) return EA_ERR_INVALID;
    *kernel = sim->kernel;
    return EA_OK;
}

ea_status ea_get_launch_count(const ea_sim *sim, uint64_t *n)
{
    if (!sim || !n) return EA_ERR_INVALID;
    *n = sim->launches;
    return EA_OK;
}

ea_status ea_synchronize(ea_sim *sim)
{
    if (!sim) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    EA_SYNC(sim);
    return EA_OK;
}

// ---- observables ----------------------------------------------------------------------------------

static ea_status fetch_counters(ea_sim *s, size_t n)
{
    EA_CUDA(s, cudaMemcpyAsync(s->h_counters.data(), s->counters, n * sizeof(unsigned long long),
                               cudaMemcpyDeviceToHost, s->stream));
    EA_SYNC(s);
    return EA_OK;
}

ea_status ea_snapshot(ea_sim *sim, int slot)
{
    if (!sim) return EA_ERR_INVALID;
    if (slot < 0 || slot >= sim->n_slots) EA_FAIL(sim, EA_ERR_INVALID, "slot %d out of range [0,%d)", slot, sim->n_slots);
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    EA_CUDA(sim, cudaMemcpyAsync(sim->snaps + (size_t)slot * sim->N, sim->spins, (size_t)sim->N * 8,
                                 cudaMemcpyDeviceToDevice, sim->stream));
    sim->slot_set[slot] = 1;
    sim->slot_t[slot] = sim->t;
    return EA_OK;
}

ea_status ea_autocorr(ea_sim *sim, int slot, int64_t *A, double *C)
{
    if (!sim || !A) return EA_ERR_INVALID;
    if (slot < 0 || slot >= sim->n_slots) EA_FAIL(sim, EA_ERR_INVALID, "slot %d out of range [0,%d)", slot, sim->n_slots);
    if (!sim->slot_set[slot]) EA_FAIL(sim, EA_ERR_STATE, "slot %d holds no snapshot", slot);
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    EA_CUDA(sim, launch_count_spins(sim, sim->snaps + (size_t)slot * sim->N));
    ea_status rc = fetch_counters(sim, 64);
    if (rc != EA_OK) return rc;
    for (int b = 0; b < 64; ++b) {
        A[b] = sim->N - 2 * (int64_t)sim->h_counters[b];
        if (C) C[b] = (double)A[b] / (double)sim->N;
    }
    return EA_OK;
}

ea_status ea_magnetisation(ea_sim *sim, int64_t *M)
{
    if (!sim || !M) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    EA_CUDA(sim, launch_count_spins(sim, nullptr));
    ea_status rc = fetch_counters(sim, 64);
    if (rc != EA_OK) return rc;
    for (int b = 0; b < 64; ++b) M[b] = sim->N - 2 * (int64_t)sim->h_counters[b];
    return EA_OK;
}

ea_status ea_energy(ea_sim *sim, int64_t *E)
{
    if (!sim || !E) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    EA_CUDA(sim, launch_count_energy(sim));
    ea_status rc = fetch_counters(sim, 64);
    if (rc != EA_OK) return rc;
    for (int b = 0; b < 64; ++b) E[b] = -3 * sim->N + 2 * (int64_t)sim->h_counters[b];
    return EA_OK;
}

ea_status ea_c4(ea_sim *sim, int r_max, int64_t *B, int64_t *q, double *c4_avg)
{
    if (!sim || !B) return EA_ERR_INVALID;
    if (sim->n_replicas != 2) EA_FAIL(sim, EA_ERR_STATE, "ea_c4 needs a 2-replica sim");
    if (r_max < 0 || r_max > sim->lat.L / 2) EA_FAIL(sim, EA_ERR_INVALID, "r_max %d outside [0, L/2]", r_max);
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    EA_CUDA(sim, launch_count_c4(sim, r_max));
    const size_t n_r = (size_t)r_max + 1, jobs = 3 * n_r + 1;
    ea_status rc = fetch_counters(sim, jobs * 32);
    if (rc != EA_OK) return rc;
    for (size_t k = 0; k < 3 * n_r * 32; ++k) B[k] = sim->N - 2 * (int64_t)sim->h_counters[k];
    if (q)
        for (int b = 0; b < 32; ++b) q[b] = sim->N - 2 * (int64_t)sim->h_counters[3 * n_r * 32 + b];
    if (c4_avg)
        for (size_t r = 0; r < n_r; ++r) {
            int64_t sum = 0; // integer sum first, one division (C-A10)
            for (int d = 0; d < 3; ++d)
                for (int b = 0; b < 32; ++b) sum += B[(d * n_r + r) * 32 + b];
            c4_avg[r] = (double)sum / (3.0 * 32.0 * (double)sim->N);
        }
    return EA_OK;
}

ea_status ea_measure(ea_sim *sim, int slot, int r_max, int64_t *A, int64_t *B, int64_t *q, int64_t *E, int64_t *M)
{
    if (!sim) return EA_ERR_INVALID;
    if (A) {
        if (slot < 0 || slot >= sim->n_slots) EA_FAIL(sim, EA_ERR_INVALID, "slot %d out of range [0,%d)", slot, sim->n_slots);
        if (!sim->slot_set[slot]) EA_FAIL(sim, EA_ERR_STATE, "slot %d holds no snapshot", slot);
    }
    if (B || q) {
        if (!B) EA_FAIL(sim, EA_ERR_INVALID, "q without B");
        if (sim->n_replicas != 2) EA_FAIL(sim, EA_ERR_STATE, "C_4 needs a 2-replica sim");
        if (r_max < 0 || r_max > sim->lat.L / 2) EA_FAIL(sim, EA_ERR_INVALID, "r_max %d outside [0, L/2]", r_max);
    }
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    // counter regions: [C_4: 3 (r_max + 1) x 32, overlap 32] [A 64] [E 64] [M 64]; all kernels enqueued, then ONE copy and sync
    const size_t n_r = (size_t)(B ? r_max + 1 : 0), c4_words = B ? (3 * n_r + 1) * 32 : 0;
    const size_t off_A = (c4_words + 63) & ~(size_t)63, off_E = off_A + 64, off_M = off_E + 64, total = off_M + 64;
    if (total > sim->n_counters) EA_FAIL(sim, EA_ERR_STATE, "counter space exhausted");
    if (B) EA_CUDA(sim, launch_count_c4(sim, r_max));
    if (A) EA_CUDA(sim, launch_count_spins(sim, sim->snaps + (size_t)slot * sim->N, sim->counters + off_A));
    if (E) EA_CUDA(sim, launch_count_energy(sim, sim->counters + off_E));
    if (M) EA_CUDA(sim, launch_count_spins(sim, nullptr, sim->counters + off_M));
    ea_status rc = fetch_counters(sim, total);
    if (rc != EA_OK) return rc;
    const unsigned long long *h = sim->h_counters.data();
    if (B) for (size_t k = 0; k < 3 * n_r * 32; ++k) B[k] = sim->N - 2 * (int64_t)h[k];
    if (q) for (int b = 0; b < 32; ++b) q[b] = sim->N - 2 * (int64_t)h[3 * n_r * 32 + b];
    if (A) for (int b = 0; b < 64; ++b) A[b] = sim->N - 2 * (int64_t)h[off_A + b];
    if (E) for (int b = 0; b < 64; ++b) E[b] = -3 * sim->N + 2 * (int64_t)h[off_E + b];
    if (M) for (int b = 0; b < 64; ++b) M[b] = sim->N - 2 * (int64_t)h[off_M + b];
    return EA_OK;
}

ea_status ea_c4_vectors(ea_sim *sim, int64_t n_vec, const int32_t *dxyz, int64_t *B)
{
    if (!sim || n_vec < 0 || (n_vec && (!dxyz || !B))) return EA_ERR_INVALID;
    if (sim->n_replicas != 2) EA_FAIL(sim, EA_ERR_STATE, "ea_c4_vectors needs a 2-replica sim");
    if (!c4_vectors_supported(sim->lat.L)) EA_FAIL(sim, EA_ERR_INVALID, "ea_c4_vectors: L must be <= 32, 64 or 128");
    if (n_vec > EA_C4_MAX_VECTORS) EA_FAIL(sim, EA_ERR_INVALID, "ea_c4_vectors: n_vec %lld > %lld", (long long)n_vec, (long long)EA_C4_MAX_VECTORS);
    DeviceGuard g(sim->device);
    try { // host buffers are sized by the caller's n_vec: no exception may cross the C ABI
        std::vector<unsigned long long> cnt((size_t)n_vec * 32);
        EA_CUDA(sim, fold_ensure_unfolded(sim));
        EA_CUDA(sim, c4_vector_counts(sim, (size_t)n_vec, dxyz, cnt.data()));
        EA_SYNC(sim);
        for (size_t k = 0; k < cnt.size(); ++k) B[k] = sim->N - 2 * (int64_t)cnt[k];
    } catch (const std::exception &) {
        EA_FAIL(sim, EA_ERR_NOMEM, "ea_c4_vectors: host allocation failed");
    }
    return EA_OK;
}

ea_status ea_c4_vectors_static(ea_sim *sim, int64_t n_vec, const int32_t *dxyz, int64_t *B)
{
    if (!sim || n_vec < 0 || (n_vec && (!dxyz || !B))) return EA_ERR_INVALID;
    if (sim->n_replicas != 2) EA_FAIL(sim, EA_ERR_STATE, "ea_c4_vectors_static needs a 2-replica sim");
    if (!c4_vectors_supported(sim->lat.L)) EA_FAIL(sim, EA_ERR_INVALID, "ea_c4_vectors_static: L must be <= 32, 64 or 128");
    if (EA_C4_STATIC_MAX_VECTORS != (int64_t)c4_vectors_static_max()) EA_FAIL(sim, EA_ERR_STATE, "ea_c4_vectors_static: header and library disagree on the limit");
    if (n_vec > EA_C4_STATIC_MAX_VECTORS)
        EA_FAIL(sim, EA_ERR_INVALID, "ea_c4_vectors_static: n_vec %lld exceeds the %lld vectors the static scratch array holds; use ea_c4_vectors",
                (long long)n_vec, (long long)EA_C4_STATIC_MAX_VECTORS);
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    // the counts land in the caller's B (same width) and are turned into sums in place: no host buffer of our own
    unsigned long long *cnt = (unsigned long long *)B;
    EA_CUDA(sim, c4_vector_counts_static(sim, (size_t)n_vec, dxyz, cnt));
    EA_SYNC(sim);
    for (size_t k = 0; k < (size_t)n_vec * 32; ++k) B[k] = sim->N - 2 * (int64_t)cnt[k];
    return EA_OK;
}

ea_status ea_c4_shells(ea_sim *sim, int r_max, int64_t *S, int64_t *mult)
{
    if (!sim || !S || !mult) return EA_ERR_INVALID;
    if (sim->n_replicas != 2) EA_FAIL(sim, EA_ERR_STATE, "ea_c4_shells needs a 2-replica sim");
    if (r_max < 0 || r_max > sim->lat.L / 2) EA_FAIL(sim, EA_ERR_INVALID, "r_max %d outside [0, L/2]", r_max);
    if (!c4_vectors_supported(sim->lat.L)) EA_FAIL(sim, EA_ERR_INVALID, "ea_c4_shells: L must be <= 32, 64 or 128");
    // B(r) = B(-r): the device visits one vector of every +-r pair (the half space dz > 0, or dz = 0 and dy > 0,
    // or dz = dy = 0 and dx > 0) and the shell receives it twice; r = 0 is B = N exactly
    try { // no exception may cross the C ABI
        std::vector<int32_t> vec;
        for (int dz = 0; dz <= r_max; ++dz)
            for (int dy = (dz ? -r_max : 0); dy <= r_max; ++dy)
                for (int dx = ((dz || dy) ? -r_max : 1); dx <= r_max; ++dx) {
                    vec.push_back(dx); vec.push_back(dy); vec.push_back(dz);
                }
        const size_t n = vec.size() / 3, n_bins = (size_t)3 * r_max * r_max + 1;
        std::vector<unsigned long long> cnt(n * 32);
        {
            DeviceGuard g(sim->device);
            EA_CUDA(sim, fold_ensure_unfolded(sim));
            EA_CUDA(sim, c4_vector_counts(sim, n, vec.data(), cnt.data()));
            EA_SYNC(sim);
        }
        for (size_t k = 0; k < n_bins * 32; ++k) S[k] = 0;
        for (size_t k = 0; k < n_bins; ++k) mult[k] = 0;
        for (int b = 0; b < 32; ++b) S[b] = sim->N;
        mult[0] = 1;
        for (size_t v = 0; v < n; ++v) {
            const int64_t d2 = (int64_t)vec[3 * v] * vec[3 * v] + (int64_t)vec[3 * v + 1] * vec[3 * v + 1] + (int64_t)vec[3 * v + 2] * vec[3 * v + 2];
            for (int b = 0; b < 32; ++b) S[d2 * 32 + b] += 2 * (sim->N - 2 * (int64_t)cnt[v * 32 + b]);
            mult[d2] += 2;
        }
    } catch (const std::exception &) {
        EA_FAIL(sim, EA_ERR_NOMEM, "ea_c4_shells: host allocation failed");
    }
    return EA_OK;
}

ea_status ea_c4_curve(const int64_t *S, const int64_t *mult, int n_bins, int n_samples, int64_t N, int r_lim,
                      int *n_pts, double *r, double *c, double *e)
{
    if (!S || !mult || !n_pts || !r || !c || !e || n_bins < 1 || n_samples < 2 || N < 1 || r_lim < 0) return EA_ERR_INVALID;
    int n = 0;
    for (int d2 = 0; d2 < n_bins; ++d2) {
        if (mult[d2] == 0 || (int64_t)d2 > (int64_t)r_lim * r_lim) continue;
        const double denom = (double)mult[d2] * (double)N;
        double sum = 0.0;
        for (int b = 0; b < n_samples; ++b) sum += (double)S[(size_t)d2 * n_samples + b] / denom;
        const double mean = sum / n_samples;
        double ss = 0.0;
        for (int b = 0; b < n_samples; ++b) {
            const double d = (double)S[(size_t)d2 * n_samples + b] / denom - mean;
            ss += d * d;
        }
        r[n] = sqrt((double)d2);
        c[n] = mean;
        e[n] = sqrt(ss / ((double)n_samples * (double)(n_samples - 1)));
        ++n;
    }
    *n_pts = n;
    return EA_OK;
}

ea_status ea_integral_estimator(int n, const double *r, const double *c, const double *e, int k, double out[4])
{
    if (n < 1 || !r || !c || !e || !out || k < 0) return EA_ERR_INVALID;
    int n_use = n;
    for (int j = 1; j < n; ++j)
        if (c[j] < 3.0 * e[j]) { n_use = j; break; }
    for (int m = 0; m < 2; ++m) {
        const int kk = k + m;
        double acc = 0.0;
        for (int j = 0; j + 1 < n_use; ++j)
            acc += 0.5 * (pow(r[j], kk) * c[j] + pow(r[j + 1], kk) * c[j + 1]) * (r[j + 1] - r[j]);
        out[m] = acc;
    }
    out[2] = out[0] != 0.0 ? out[1] / out[0] : NAN;
    out[3] = r[n_use - 1];
    return EA_OK;
}

// ---- canonical packed I/O ---------------------------------------------------------------------------

ea_status ea_get_spins(ea_sim *sim, uint64_t *host)
{
    if (!sim || !host) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    EA_CUDA(sim, fold_ensure_unfolded(sim));
    EA_CUDA(sim, launch_unpack_spins(sim, sim->spins, sim->stage));
    EA_CUDA(sim, cudaMemcpyAsync(host, sim->stage, (size_t)sim->N * 8, cudaMemcpyDeviceToHost, sim->stream));
    EA_SYNC(sim);
    return EA_OK;
}

ea_status ea_get_snapshot(ea_sim *sim, int slot, uint64_t *host)
{
    if (!sim || !host) return EA_ERR_INVALID;
    if (slot < 0 || slot >= sim->n_slots) EA_FAIL(sim, EA_ERR_INVALID, "slot %d out of range [0,%d)", slot, sim->n_slots);
    if (!sim->slot_set[slot]) EA_FAIL(sim, EA_ERR_STATE, "slot %d holds no snapshot", slot);
    DeviceGuard g(sim->device);
    EA_CUDA(sim, launch_unpack_spins(sim, sim->snaps + (size_t)slot * sim->N, sim->stage));
    EA_CUDA(sim, cudaMemcpyAsync(host, sim->stage, (size_t)sim->N * 8, cudaMemcpyDeviceToHost, sim->stream));
    EA_SYNC(sim);
    return EA_OK;
}

ea_status ea_set_spins(ea_sim *sim, const uint64_t *host)
{
    if (!sim || !host) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    EA_CUDA(sim, cudaMemcpyAsync(sim->stage, host, (size_t)sim->N * 8, cudaMemcpyHostToDevice, sim->stream));
    EA_CUDA(sim, launch_pack_spins(sim, sim->stage, sim->spins));
    if (sim->n_samples < EA_LANES) EA_CUDA(sim, fold_from_standard(sim, true, false)); // unused lanes are dropped
    EA_SYNC(sim);
    return EA_OK;
}

ea_status ea_get_bonds(ea_sim *sim, uint64_t *host)
{
    if (!sim || !host) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    for (int d = 0; d < 3; ++d) {
        EA_CUDA(sim, launch_unpack_bonds(sim, d, sim->stage));
        EA_CUDA(sim, cudaMemcpyAsync(host + (size_t)d * sim->N, sim->stage, (size_t)sim->N * 8, cudaMemcpyDeviceToHost,
                                     sim->stream)); // stream order keeps unpack d+1 behind this copy of the staging buffer
    }
    EA_SYNC(sim);
    return EA_OK;
}

ea_status ea_set_bonds(ea_sim *sim, const uint64_t *host)
{
    if (!sim || !host) return EA_ERR_INVALID;
    DeviceGuard g(sim->device);
    // both replicas have "the same bond configuration": the pack kernel raises a flag on hi != lo
    unsigned *d_bad = sim->resident_flags + (resident_flag_bytes() / sizeof(unsigned) - 31);
    EA_CUDA(sim, cudaMemsetAsync(d_bad, 0, sizeof(unsigned), sim->stream));
    for (int d = 0; d < 3; ++d) { // the staging buffer holds one direction; stream order keeps copy d+1 behind pack d
        EA_CUDA(sim, cudaMemcpyAsync(sim->stage, host + (size_t)d * sim->N, (size_t)sim->N * 8, cudaMemcpyHostToDevice,
                                     sim->stream));
        EA_CUDA(sim, launch_pack_bonds(sim, d, sim->stage, d_bad));
    }
    if (sim->n_samples < EA_LANES) EA_CUDA(sim, fold_from_standard(sim, false, true));
    unsigned bad = 0;
    EA_CUDA(sim, cudaMemcpyAsync(&bad, d_bad, sizeof(bad), cudaMemcpyDeviceToHost, sim->stream));
    EA_SYNC(sim);
    if (bad)
        EA_FAIL(sim, EA_ERR_INVALID, "2-replica sim: a bond word has hi half != lo half; the sim's bonds are now undefined, set them again");
    return EA_OK;
}

/* Host-only consistency checks (no device): the RESIDENT row schedules. */
ea_status ea_selftest_host(void) { return resident_tables_ok() ? EA_OK : EA_ERR_STATE; }

// ---- batches of small sims (one launch per colour for all of them) ---------------------------------

struct ea_batch {
    std::vector<ea_sim *> sims;
    int L = 0, n_replicas = 0, device = 0;
    cudaStream_t stream = nullptr; // the first sim's stream
    char *d_args = nullptr;        // [2][K] launch arguments (parity-major)
    uint64_t **d_times = nullptr;  // [K] the sims' device clocks
    cudaEvent_t ev = nullptr;
    cudaGraphExec_t graph_exec = nullptr;
    bool graph_always = false, graph_hb = false;
    std::vector<char> h_args;
};

static void batch_free(ea_batch *b)
{
    if (b->graph_exec) cudaGraphExecDestroy(b->graph_exec);
    if (b->d_args) cudaFree(b->d_args);
    if (b->d_times) cudaFree(b->d_times);
    if (b->ev) cudaEventDestroy(b->ev);
    delete b;
}

ea_status ea_batch_create(ea_sim *const *sims, int n_sims, ea_batch **out)
{
    if (!sims || !out || n_sims < 1 || n_sims > 65535) return EA_ERR_INVALID;
    for (int i = 0; i < n_sims; ++i) {
        if (!sims[i]) return EA_ERR_INVALID;
        for (int j = 0; j < i; ++j)
            if (sims[j] == sims[i]) return EA_ERR_INVALID;
        if (sims[i]->lat.L != sims[0]->lat.L || sims[i]->n_replicas != sims[0]->n_replicas || sims[i]->device != sims[0]->device ||
            sims[i]->n_samples != EA_LANES)
            EA_FAIL(sims[i], EA_ERR_INVALID, "a batch needs sims of one L, one replica mode, 64 samples, one device");
    }
    if (!rows_persistent_valid(sims[0]->lat.L)) EA_FAIL(sims[0], EA_ERR_INVALID, "batches are for L = 16, 32, 64 (larger lattices fill the device alone)");
    ea_batch *b = new (std::nothrow) ea_batch();
    if (!b) return EA_ERR_NOMEM;
    b->sims.assign(sims, sims + n_sims);
    b->L = sims[0]->lat.L;
    b->n_replicas = sims[0]->n_replicas;
    b->device = sims[0]->device;
    b->stream = sims[0]->stream;
    DeviceGuard g(b->device);
    const size_t K = (size_t)n_sims;
    std::vector<uint64_t *> h_times(K);
    for (size_t i = 0; i < K; ++i) h_times[i] = sims[i]->d_time;
    b->h_args.resize(2 * K * batch_args_bytes());
    if (cudaMalloc((void **)&b->d_args, b->h_args.size()) != cudaSuccess || cudaMalloc((void **)&b->d_times, K * sizeof(uint64_t *)) != cudaSuccess ||
        cudaEventCreateWithFlags(&b->ev, cudaEventDisableTiming) != cudaSuccess ||
        cudaMemcpy(b->d_times, h_times.data(), K * sizeof(uint64_t *), cudaMemcpyHostToDevice) != cudaSuccess) {
        batch_free(b);
        return EA_ERR_NOMEM;
    }
    *out = b;
    return EA_OK;
}

ea_status ea_batch_destroy(ea_batch *b)
{
    if (!b) return EA_OK;
    DeviceGuard g(b->device);
    cudaStreamSynchronize(b->stream);
    batch_free(b);
    return EA_OK;
}

static cudaError_t batch_half_sweeps(ea_batch *b, bool always, bool hb, uint32_t k)
{
    const unsigned K = (unsigned)b->sims.size();
    const char *a0 = b->d_args, *a1 = b->d_args + (size_t)K * batch_args_bytes();
    cudaError_t e = launch_half_sweep_batch(b->L, b->n_replicas, always, hb, a0, K, k, b->stream);
    if (e == cudaSuccess) e = launch_half_sweep_batch(b->L, b->n_replicas, always, hb, a1, K, k, b->stream);
    return e;
}

ea_status ea_batch_sweep(ea_batch *b, uint64_t n)
{
    if (!b) return EA_ERR_INVALID;
    ea_sim *s0 = b->sims[0];
    const size_t K = b->sims.size(), az = batch_args_bytes();
    bool always = false;
    const bool hb = s0->dynamics == EA_DYN_HEATBATH;
    for (ea_sim *s : b->sims) {
        if (s->dynamics != s0->dynamics) EA_FAIL(s0, EA_ERR_STATE, "the sims of a batch must share the dynamics");
        always |= (s->th.always[0] | s->th.always[1] | s->th.always[2]) != 0;
    }
    if (!n) return EA_OK;
    DeviceGuard g(b->device);
    for (size_t i = 0; i < K; ++i) { // temperatures may have changed: the arguments are rebuilt every call
        fill_batch_args(b->sims[i], 0, b->h_args.data() + i * az);
        fill_batch_args(b->sims[i], 1, b->h_args.data() + (K + i) * az);
    }
    for (size_t i = 1; i < K; ++i) // the batch runs on the first sim's stream, behind whatever the others have queued
        if (b->sims[i]->stream != b->stream) {
            EA_CUDA(s0, cudaEventRecord(b->ev, b->sims[i]->stream));
            EA_CUDA(s0, cudaStreamWaitEvent(b->stream, b->ev, 0));
        }
    EA_CUDA(s0, cudaMemcpyAsync(b->d_args, b->h_args.data(), b->h_args.size(), cudaMemcpyHostToDevice, b->stream));
    for (ea_sim *s : b->sims) EA_CUDA(s0, cudaMemcpyAsync(s->d_time, &s->t, 8, cudaMemcpyHostToDevice, b->stream));
    uint64_t left = n;
    if (left >= (uint64_t)GRAPH_SWEEPS) {
        if (!b->graph_exec || b->graph_always != always || b->graph_hb != hb) {
            if (b->graph_exec) cudaGraphExecDestroy(b->graph_exec);
            b->graph_exec = nullptr;
            cudaGraph_t graph = nullptr;
            EA_CUDA(s0, cudaStreamBeginCapture(b->stream, cudaStreamCaptureModeThreadLocal));
            cudaError_t e = cudaSuccess;
            for (int k = 0; k < GRAPH_SWEEPS && e == cudaSuccess; ++k) e = batch_half_sweeps(b, always, hb, (uint32_t)k);
            if (e == cudaSuccess) e = launch_bump_time_batch(b->d_times, (unsigned)K, GRAPH_SWEEPS, b->stream);
            cudaError_t e2 = cudaStreamEndCapture(b->stream, &graph);
            if (e != cudaSuccess || e2 != cudaSuccess) {
                if (graph) cudaGraphDestroy(graph);
                EA_FAIL(s0, EA_ERR_CUDA, "batch graph capture: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
            }
            e = cudaGraphInstantiate(&b->graph_exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { b->graph_exec = nullptr; EA_FAIL(s0, EA_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e)); }
            b->graph_always = always;
            b->graph_hb = hb;
        }
        while (left >= (uint64_t)GRAPH_SWEEPS) {
            const cudaError_t e = cudaGraphLaunch(b->graph_exec, b->stream);
            if (e != cudaSuccess) { // the members' clocks count the replays that were queued
                for (ea_sim *s : b->sims) s->t += n - left;
                EA_FAIL(s0, EA_ERR_CUDA, "cudaGraphLaunch: %s", cudaGetErrorString(e));
            }
            s0->count_launch(2 * GRAPH_SWEEPS + 1);
            left -= GRAPH_SWEEPS;
        }
    }
    for (ea_sim *s : b->sims) s->t += n - left;
    if (left) { // a failure in here leaves the members' spins part-way through these `left` sweeps (undefined)
        for (uint32_t k = 0; k < (uint32_t)left; ++k) EA_CUDA(s0, batch_half_sweeps(b, always, hb, k));
        EA_CUDA(s0, launch_bump_time_batch(b->d_times, (unsigned)K, (uint32_t)left, b->stream));
        s0->count_launch(2 * (unsigned)left + 1);
        for (ea_sim *s : b->sims) s->t += left;
    }
    EA_CUDA(s0, cudaEventRecord(b->ev, b->stream)); // later calls on the other sims' streams see the batch's work
    for (size_t i = 1; i < K; ++i)
        if (b->sims[i]->stream != b->stream) EA_CUDA(s0, cudaStreamWaitEvent(b->sims[i]->stream, b->ev, 0));
    return EA_OK;
}

ea_status ea_selftest_pipes(int device, double out[8])
{
    if (!out) return EA_ERR_INVALID;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) return EA_ERR_CUDA;
    if (device < 0 && cudaGetDevice(&device) != cudaSuccess) return EA_ERR_CUDA;
    if (device >= n_dev) return EA_ERR_INVALID;
    DeviceGuard g(device);
    if (!g.ok) return EA_ERR_CUDA;
    double r[8];
    if (pipe_rates(device, r) != cudaSuccess) return EA_ERR_CUDA;
    memcpy(out, r, sizeof(r));
    return EA_OK;
}

ea_status ea_philox_selftest(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    if (!ctr || !key || !out) return EA_ERR_INVALID;
    return philox_selftest(ctr, key, out) == cudaSuccess ? EA_OK : EA_ERR_CUDA;
}

} // extern "C"

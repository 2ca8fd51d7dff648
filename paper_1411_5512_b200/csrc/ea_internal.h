// ea_internal.h -- host-side state of one sim and the launch wrappers of the kernels (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/ea.h"
#include "ea_device.cuh"

struct ea_sim {
    ea::Lattice lat;
    int64_t N = 0;
    int n_replicas = 1, n_slots = 0;
    int n_samples = 64;           // M: samples per word; < 64 = mixed multispin coding (ea_fold.cu), K = 64 / M slabs
    uint64_t *f_spins = nullptr;  // folded spins [2][Nh/K]: the state the sweeps run on when M < 64
    uint64_t *f_bonds = nullptr;  // folded bonds [2][3][Nh/K], 64-bit words
    bool unfolded_valid = true;   // M < 64: does `spins` (standard layout, unused lanes zero) mirror f_spins?
    double p = 0, T = 0;
    uint64_t seed = 0, t = 0;
    uint64_t thr[3] = {0, 0, 0};
    ea::Thresholds th;
    int device = 0;
    int n_sm = 148;
    cudaStream_t stream = nullptr;
    int kernel = EA_KERNEL_SCALAR; // resolved variant
    int dynamics = EA_DYN_METROPOLIS;
    int n_concurrent = 1;         // ea_set_concurrency_hint
    uint64_t thr_hb[7] = {0, 0, 0, 0, 0, 0, 0};

    bool own_ws = false, own_stream = false;
    char *ws = nullptr;
    size_t ws_bytes = 0;
    uint64_t *spins = nullptr;    // [2][Nh]
    void *bonds = nullptr;        // BondT [2][3][Nh]
    uint64_t *snaps = nullptr;    // [n_slots][2][Nh]
    uint64_t *stage = nullptr;    // [N] canonical staging for get/set
    unsigned long long *counters = nullptr; // [n_counters]
    size_t n_counters = 0;
    std::vector<char> slot_set;
    std::vector<uint64_t> slot_t;
    std::vector<unsigned long long> h_counters;

    // CUDA graph of a block of sweeps (launch-bound small lattices)
    cudaGraphExec_t graph_exec = nullptr;
    int graph_sweeps = 0;
    int graph_kernel = -1;
    uint64_t *d_time = nullptr;   // device copy of t consumed by graph-launched kernels

    // RESIDENT kernel (L = 128): per-CTA step flags + abort word in the workspace, and the flag epoch
    unsigned *resident_flags = nullptr;
    uint32_t resident_epoch = 0;
    int resident_tiles = 0;           // CTAs of the partition whose tile table sits behind the flags (0: none)
    uint64_t resident_min_sweeps = 1; // shorter ea_sweep calls use the ROWS launches (AUTO: 8; SMALL under AUTO: 2)
    bool resident_used = false;       // a resident launch is in flight / unchecked: see check_resident()
    uint64_t resident_timeout_ns = 20000000000ull; // neighbour wait gives up after this (EA_RESIDENT_TIMEOUT_MS)

    // grow-only scratch of ea_c4_vectors / ea_c4_shells (job list, per-vector counters), owned by the sim
    void *c4v_jobs = nullptr;
    size_t c4v_jobs_bytes = 0;
    unsigned long long *c4v_out = nullptr;
    size_t c4v_out_bytes = 0;

    // kernels this sim has put on the device (a graph replay counts its kernel nodes); bench.py's gpu_launches
    uint64_t launches = 0;
    bool capturing = false;
    void count_launch(unsigned n = 1) { if (!capturing) launches += n; }

    std::string err;

    int bond_bytes() const { return n_replicas == 2 ? 4 : 8; }
    uint64_t *spins_c(int c) const { return spins + (size_t)c * lat.Nh; }
};

namespace ea {

struct WorkspaceLayout {
    size_t off_spins, off_bonds, off_snaps, off_stage, off_counters, off_time, off_flags, off_fold, total;
    size_t n_counters;
};
WorkspaceLayout workspace_layout(int L, int n_samples, int n_replicas, int n_slots);

// ---- launch wrappers (each returns the cudaError_t of the launch) -------------------------------
cudaError_t launch_init_spins(ea_sim *s);
cudaError_t launch_init_bonds(ea_sim *s);
// one colour of sweep t.  If d_time != nullptr the kernels read t = *d_time + t_offset on the device.
cudaError_t launch_half_sweep(ea_sim *s, int parity, uint64_t t, const uint64_t *d_time, uint32_t t_offset,
                              cudaStream_t st);
cudaError_t launch_bump_time(ea_sim *s, uint32_t n, cudaStream_t st);
// mixed multispin coding, M < 64 samples per word (ea_fold.cu)
bool fold_valid(int L, int n_samples, int n_replicas);
size_t fold_bytes(int L, int n_samples);
uint64_t expand_lanes_host(const ea_sim *s);                     // the 64-lane mask of the samples carried
cudaError_t fold_from_standard(ea_sim *s, bool spins, bool bonds); // mask unused lanes, (re)build the folded copies
cudaError_t fold_ensure_unfolded(ea_sim *s);                     // refresh `spins` from f_spins if stale
cudaError_t launch_half_sweep_fold(ea_sim *s, int parity, uint64_t t, const uint64_t *d_time, uint32_t t_offset,
                                   cudaStream_t st);
// BATCH (ea_sweep.cu): K small sims per launch, blockIdx.y = sim
void fill_batch_args(const ea_sim *s, int parity, void *out);
size_t batch_args_bytes();
cudaError_t launch_half_sweep_batch(int L, int n_replicas, bool always, bool heatbath, const void *d_args, unsigned n_sims,
                                    uint32_t t_offset, cudaStream_t st);
cudaError_t launch_bump_time_batch(uint64_t *const *d_times, unsigned n_sims, uint32_t n, cudaStream_t st);
// ROWS_PERSISTENT (ea_sweep.cu; L = 16, 32, 64): n sweeps in one cooperative launch with a grid barrier per colour
bool rows_persistent_valid(int L);
cudaError_t launch_sweeps_rows_persistent(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st);
// SMALL (ea_sweep_small.cu; L % 4 == 0, L <= 32): n sweeps in one launch, lattice resident in the shared memory of one
// CTA or one thread-block cluster
int small_cluster_size(int L, int n_replicas); // 0: not valid for this shape
bool small_supported(const ea_sim *s, std::string *why = nullptr);
cudaError_t launch_sweeps_small(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st);
// RESIDENT (ea_sweep_resident.cu): n sweeps from sweep index t0 in one cooperative launch
bool resident_supported(const ea_sim *s, std::string *why = nullptr);
size_t resident_flag_bytes();   // flag lines + abort line
size_t resident_aux_bytes();    // flags + the tile table behind them (workspace)
cudaError_t resident_prepare(ea_sim *s, std::string *why = nullptr); // build + upload the tile table (stream-ordered)
bool resident_tables_ok();
cudaError_t launch_sweeps_resident(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st);

// canonical <-> internal
cudaError_t launch_pack_spins(ea_sim *s, const uint64_t *d_canon, uint64_t *d_internal);   // canonical -> internal
cudaError_t launch_unpack_spins(ea_sim *s, const uint64_t *d_internal, uint64_t *d_canon); // internal -> canonical
cudaError_t launch_pack_bonds(ea_sim *s, int d, const uint64_t *d_canon, unsigned *d_bad); // one direction, N words; *d_bad |= 1 if hi != lo (2 replicas)
cudaError_t launch_unpack_bonds(ea_sim *s, int d, uint64_t *d_canon);

// observables: per-sample bit counts into s->counters (zeroed by the wrapper)
// (dst: 64 counters; nullptr = s->counters)
cudaError_t launch_count_spins(ea_sim *s, const uint64_t *d_other /* nullable: XOR partner, same layout */, unsigned long long *dst = nullptr);
cudaError_t launch_count_energy(ea_sim *s, unsigned long long *dst = nullptr);
cudaError_t launch_count_c4(ea_sim *s, int r_max); // counters[(d*(r_max+1)+r)*32+b], then [3*(r_max+1)*32 + b] = overlap

// full-vector C_4 (ea_c4_vectors.cu): per-sample counts of q_i != q_{i+r} for n lattice vectors; host result
bool c4_vectors_supported(int L);
cudaError_t c4_vector_counts(ea_sim *s, size_t n, const int32_t *vec, unsigned long long *counts);
size_t c4_vectors_static_max();
cudaError_t c4_vector_counts_static(ea_sim *s, size_t n, const int32_t *vec, unsigned long long *counts); // no allocation; n <= c4_vectors_static_max()

cudaError_t pipe_rates(int device, double out[8]);
cudaError_t philox_selftest(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

} // namespace ea

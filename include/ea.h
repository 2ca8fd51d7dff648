/*
 * ea.h -- C ABI of libea_b200.so: checkerboard Metropolis sweeps of the 3D +-J
 * Edwards-Anderson model, 64 samples multispin-coded per 64-bit word, and the popcount
 * observables C(t,t_w), C_4(r,t_w), energy, magnetisation -- hand-written sm_100a kernels.
 *
 * Paper: Manssen & Hartmann, arXiv:1411.5512; citations are PAPER.md:<line> + section/equation.
 * "C-xx" are the readings of the paper listed in DESIGN.md section 2 (the stream contract).
 *
 * Conventions for every entry point
 *   - Plain C types only.  "host" pointers are caller-allocated host memory, "device" pointers
 *     are CUDA device memory.  Nothing allocated by the library is ever handed to the caller.
 *   - Every function returns an ea_status; on any error the outputs are untouched and
 *     ea_last_error(sim) holds a message.  No exceptions or aborts cross the boundary.
 *   - ea_sweep / ea_snapshot are asynchronous on the sim's stream; every call that returns
 *     host data synchronises that stream before returning.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - After EA_ERR_CUDA from a call that advances the dynamics the spin state is undefined (the device may
 *     have run part of the request); t counts the sweeps whose launches were all queued.
 *   - Results depend only on (L, p, T, n_replicas, seed, t): never on the GPU, the kernel
 *     variant or the launch geometry.  ea_sweep(a); ea_sweep(b) == ea_sweep(a+b).
 *   - There is no CPU fallback: without a CUDA device every compute call returns EA_ERR_CUDA.
 *
 * Canonical host format (the exchange format of ea_get_* / ea_set_*; C-A1, C-A2):
 *   site = x + L*(y + L*z);  spins[site] : bit b = 1 <-> S = -1 of sample b;
 *   bonds[d*N + site], d = 0,1,2 : bond between site and site + e_d (+x,+y,+z, periodic),
 *   bit b = 1 <-> J = -1 of sample b.  n_replicas == 2: sample b (<32) = disorder b replica (a),
 *   sample b+32 = disorder b replica (b); every bond word has hi half == lo half.
 */
#ifndef EA_B200_H
#define EA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EA_LANES 64 /* samples per multispin word (III) */
#define EA_C4_MAX_VECTORS ((int64_t)1 << 24) /* ea_c4_vectors: most vectors per call (a full L = 128 torus has 2^21) */
#define EA_C4_STATIC_MAX_VECTORS ((int64_t)1024) /* ea_c4_vectors_static: most vectors per call */

typedef struct ea_sim ea_sim; /* opaque; one batch of 64 samples on one L^3 lattice */

typedef enum {
    EA_OK = 0,
    EA_ERR_INVALID = 1, /* bad argument (see each call)                                   */
    EA_ERR_CUDA = 2,    /* CUDA runtime error, or no device                                */
    EA_ERR_NOMEM = 3,   /* host or device allocation failed / workspace too small          */
    EA_ERR_STATE = 4    /* call not valid in this state (unset slot, c4 on 1 replica, ...) */
} ea_status;

/* Sweep kernel variants (all bit-identical; selection is a performance matter only). */
typedef enum {
    EA_KERNEL_AUTO = 0,   /* the fastest variant valid for L                              */
    EA_KERNEL_SCALAR = 1, /* one site per thread, 64-bit loads; any even L >= 2           */
    EA_KERNEL_VEC2 = 2,   /* two sites per thread, 128-bit loads; L % 4 == 0              */
    EA_KERNEL_ROWS = 3,   /* warp marches along y with a register window; L % 4 == 0      */
    EA_KERNEL_RESIDENT = 4, /* persistent cooperative kernel, many sweeps per launch (L = 128): 148 tiles on a 148-SM part,
                               128 otherwise; needs a device with cooperative launch, >= 128 SMs and 170 (185) KB of
                               shared memory per CTA (ea_last_error / stderr say which is missing).  Its CTAs wait for their neighbours' step flags; a wait
                               that sees nothing for EA_RESIDENT_TIMEOUT_MS (environment, read at ea_create;
                               default 20000) gives up, and the next synchronising call returns EA_ERR_CUDA */
    EA_KERNEL_FOLD = 5,    /* what a sim with n_samples < 64 runs (not selectable)        */
    EA_KERNEL_ROWS_PERSISTENT = 6, /* ROWS with a grid barrier per colour, one launch per ea_sweep (L = 16, 32, 64);
                                     measured slower than the graph replays, never chosen by AUTO */
    EA_KERNEL_SMALL = 7   /* small lattices (L % 4 == 0, L <= 32): spins and bonds resident in the shared memory of one
                             CTA (L <= 8) or of one thread-block cluster (L = 32: 16 CTAs; boundary planes pushed into
                             the neighbouring CTA's shared memory, an mbarrier per colour); one launch per ea_sweep.
                             AUTO uses it for ea_sweep(n >= 2); shorter calls go as per-colour launches */
} ea_kernel;

/* Single-spin dynamics.  The paper uses Metropolis (Eq. 9); heat bath is the variant of SURVEY 8(f)
 * item 4 -- reading C-HB: flip with probability 1 / (1 + exp(Delta E / T)), Delta E = 12 - 4 n_u, for every
 * n_u = 0..6 (Delta E = 0: exactly 1/2), same random numbers, same strict "<" against 32-bit thresholds. */
typedef enum { EA_DYN_METROPOLIS = 0, EA_DYN_HEATBATH = 1 } ea_dynamics;

typedef struct ea_params {
    int32_t L;          /* lattice side; even, >= 2, L^3 < 2^31 (C-A1)                     */
    int32_t n_samples;  /* M = samples per word: 64, or 32, 16, ... (mixed multispin coding, PAPER.md:94:
                           64/M z-slabs of the lattice share a word; needs L % 4 == 0 and L*M/64 even;
                           the M samples are lanes 0..M/2-1 and 32..32+M/2-1 of the 64-sample sim of
                           the same seed (2 replicas) or lanes 0..M-1 (1 replica), bit for bit: C-M.
                           Host arrays keep their 64- / 32-entry shape; unused entries are unspecified) */
    int32_t n_replicas; /* 1: 64 independent samples; 2: 32 disorders x 2 replicas (C-A2r) */
    int32_t n_slots;    /* snapshot slots for ea_snapshot / ea_autocorr (>= 0)             */
    double p;           /* P(J = +1), in [0,1]                              */
    double T;           /* temperature, >= 0; 0 and +inf legal (Eq. 9)        */
    uint64_t seed;      /* Philox key (C-A6)                                               */
    int32_t device;     /* CUDA device ordinal; -1 = current device                        */
    int32_t kernel;     /* ea_kernel                                                       */
    void *stream;       /* cudaStream_t to run on (caller-owned); NULL = the library creates and owns a
                           non-blocking stream.  The legacy default stream (cudaStreamLegacy) cannot be
                           captured into a CUDA graph and is refused with EA_ERR_INVALID                */
    void *d_workspace;  /* device memory, >= ea_workspace_bytes(...), 256-byte aligned, anywhere in the
                           address space, caller-owned and alive until ea_destroy; work queued on other
                           streams that still touches it must be complete (or ordered before `stream`)
                           when ea_create_ex is called; NULL = library allocates                         */
    size_t workspace_bytes;
} ea_params;

/* Bytes of device memory one sim needs (0 if the arguments are invalid). */
size_t ea_workspace_bytes(int L, int n_replicas, int n_slots);                 /* n_samples = 64 */
size_t ea_workspace_bytes_ex(int L, int n_samples, int n_replicas, int n_slots);

/* Create a sim: bonds iid with P(J=+1) = p per disorder sample (C-A9), spins
 * uniform +-1 (random start = quench from T = inf, C-A8), t = 0.
 * ea_create: 64 independent samples (n_samples must be 64), 2 slots, current device, own stream.
 * EA_ERR_INVALID: L odd / < 2 / too large, p outside [0,1] or NaN, T < 0 or NaN, n_samples not valid for L,
 * n_replicas not 1|2, n_slots < 0, out == NULL.  The caller owns *out until ea_destroy. */
ea_status ea_create(int L, double p, double T, int n_samples, uint64_t seed, ea_sim **out);
ea_status ea_create_ex(const ea_params *prm, ea_sim **out);
ea_status ea_destroy(ea_sim *sim);

/* n full sweeps: each = all sites with (x+y+z)&1 == 0, then all with parity 1 (C-S2),
 * single-spin-flip Metropolis with Eq. 9 (C-A4), one Philox4x32-10 block per sweep and pair of
 * x-adjacent same-colour sites, all four output words used (C-A6, C-A7).  Asynchronous; t += n. */
ea_status ea_sweep(ea_sim *sim, uint64_t n);
/* One colour only (parity 0 or 1) of sweep t; does not advance t.  For tests of the half-step. */
ea_status ea_half_sweep(ea_sim *sim, int parity);

ea_status ea_get_time(const ea_sim *sim, uint64_t *t); /* completed sweeps since the random start (C-S11) */
ea_status ea_set_time(ea_sim *sim, uint64_t t);
ea_status ea_set_temperature(ea_sim *sim, double T);   /* recomputes the thresholds               */
ea_status ea_get_thresholds(const ea_sim *sim, uint64_t thr[3]); /* thr[n_u], n_u = 0,1,2 (C-A4)  */
ea_status ea_set_dynamics(ea_sim *sim, int dynamics);  /* ea_dynamics                                          */
ea_status ea_get_dynamics(const ea_sim *sim, int *dynamics);
ea_status ea_get_thresholds_heatbath(const ea_sim *sim, uint64_t thr[7]); /* thr[n_u], n_u = 0..6 (C-HB)     */
ea_status ea_set_kernel(ea_sim *sim, int kernel);      /* EA_ERR_INVALID if not valid for this L  */
ea_status ea_get_kernel(const ea_sim *sim, int *kernel); /* the variant AUTO resolved to          */
/* How many sims the caller advances at the same time on this device (a scan), n >= 1; default 1.  Results
 * never depend on it: the library only chooses between code paths tuned for one sim alone on the device (latency) and
 * for many sims sharing its SMs (issue slots) -- today in the small-lattice kernel.  EA_ERR_INVALID if n < 1. */
ea_status ea_set_concurrency_hint(ea_sim *sim, int n_concurrent_sims);
ea_status ea_synchronize(ea_sim *sim);                 /* wait for the sim's stream               */
/* Kernels this sim has launched on the device since ea_create (a CUDA-graph replay counts its kernel nodes). */
ea_status ea_get_launch_count(const ea_sim *sim, uint64_t *n);

/* Keep sigma(t) in slot (device copy; the paper wrote configurations to disk). */
ea_status ea_snapshot(ea_sim *sim, int slot);
/* A[b] = sum_i S_i,b(t_w) S_i,b(now) = N C(t,t_w) (Eq. 7); C[b] = A[b]/N or NULL.
 * host arrays of 64.  EA_ERR_INVALID bad slot, EA_ERR_STATE unset slot. */
ea_status ea_autocorr(ea_sim *sim, int slot, int64_t *A, double *C);
/* Replica overlap and four-point correlation along the lattice axes (Eq. 2-3; C-S8):
 * q[b] = sum_i q_i, q_i = S^a_i S^b_i;  B[(d*(r_max+1) + r)*32 + b] = sum_i q_i q_{i + r e_d} = N C_4.
 * c4_avg[r] = sum_d sum_b B / (3*32*N) or NULL; q may be NULL.  0 <= r_max <= L/2.
 * EA_ERR_STATE on a 1-replica sim. */
ea_status ea_c4(ea_sim *sim, int r_max, int64_t *B, int64_t *q, double *c4_avg);
/* Four-point correlation for arbitrary lattice vectors (Eq. 3, with "i + r" read as any lattice
 * vector, periodic -- reading C-S8v; the paper's "all r >= 3" reference set, and Fig. 2):
 *   B[v*32 + b] = sum_i q_i q_{i + r_v},  r_v = (dxyz[3v], dxyz[3v+1], dxyz[3v+2]), any integers.
 * host arrays: dxyz 3 n_vec int32, B 32 n_vec int64.  EA_ERR_STATE on a 1-replica sim; EA_ERR_INVALID unless
 * L <= 32 or L in {64, 128}, or n_vec > EA_C4_MAX_VECTORS; EA_ERR_NOMEM if a host buffer cannot be allocated. */
ea_status ea_c4_vectors(ea_sim *sim, int64_t n_vec, const int32_t *dxyz, int64_t *B);
/* The same result for n_vec <= EA_C4_STATIC_MAX_VECTORS with NO allocation on the device or the host, for callers that cannot
 * call cudaMalloc (inside a stream capture, in a serving loop, under a harness that forbids it): ea_c4_vectors keeps its job
 * list and counters in grow-only cudaMalloc buffers; this call keeps them in one file-scope device array of 301 KiB (256 KiB of
 * counters, 20 KiB of jobs, 24.5 KiB for the transposed field of an L < 16 lattice) that every GPU which loads the library holds
 * until the process exits.  Same arguments, same B.  EA_ERR_INVALID with an ea_last_error text if n_vec exceeds the limit.
 * Every call on a device shares that array, which keeps the last call's contents (the call clears the counters it uses):
 * calls that overlap on the GPU -- two sims on two streams, two host threads -- race; serialise them. */
ea_status ea_c4_vectors_static(ea_sim *sim, int64_t n_vec, const int32_t *dxyz, int64_t *B);
/* Shell sums over the cube |dx|, |dy|, |dz| <= r_max (0 <= r_max <= L/2), by squared length d2 = 0 .. 3 r_max^2:
 *   S[d2*32 + b] = sum_{|r|^2 = d2} B_b(r),  mult[d2] = number of those vectors (0 for an empty shell),
 * so C_4(|r| = sqrt(d2)) = S / (mult N).  r and -r are both counted; with r_max = L/2 the components +L/2 and
 * -L/2 (one displacement on the torus) count as two vectors.  host arrays of (3 r_max^2 + 1) * 32 and 3 r_max^2 + 1. */
ea_status ea_c4_shells(ea_sim *sim, int r_max, int64_t *S, int64_t *mult);
/* Host arithmetic in double (no device work), the post-processing of PAPER.md:116 -- reading C-S12:
 * ea_c4_curve: shell sums -> points with mult > 0 and d2 <= r_lim^2, ascending: r = sqrt(d2), c = mean over the
 *   n_samples disorder samples of S/(mult N), e = its standard error sqrt(sum (c_b - c)^2 / (n (n-1))).
 *   r, c, e: host arrays of n_bins; *n_pts = points written.
 * ea_integral_estimator (Eq. 5-6): with j* the first j >= 1 where c_j < 3 e_j (the paper's cut-off,
 *   :116; all points if none), I_k = sum_{j < j*-1} (r_j^k c_j + r_{j+1}^k c_{j+1}) (r_{j+1} - r_j) / 2 (trapezoid),
 *   out = { I_k, I_{k+1}, xi_k = I_{k+1} / I_k, r_{j*-1} }.  The paper adds the tail of its fitted form (4) beyond
 *   the cut-off; fits are out of scope and no tail is added. */
ea_status ea_c4_curve(const int64_t *S, const int64_t *mult, int n_bins, int n_samples, int64_t N, int r_lim,
                      int *n_pts, double *r, double *c, double *e);
ea_status ea_integral_estimator(int n, const double *r, const double *c, const double *e, int k, double out[4]);
/* E[b] = -sum_<ij> J_ij S_i S_j over the 3N bonds (Eq. 1); host array of 64. */
ea_status ea_energy(ea_sim *sim, int64_t *E);
/* M[b] = sum_i S_i,b (C-S14); host array of 64. */
ea_status ea_magnetisation(ea_sim *sim, int64_t *M);

/* One measure point (the observables the paper took from every stored configuration) in ONE call: the same
 * numbers as ea_autocorr(slot) / ea_c4(r_max) / ea_energy / ea_magnetisation, but all kernels are enqueued back to back and
 * the host waits once (five separate calls cost five round trips, ~25 us each -- as much as the kernels at L = 128).
 * Any of A [64], B [3][r_max+1][32] (+ q [32]), E [64], M [64] may be NULL (skipped); slot / r_max are ignored when A / B is
 * NULL.  Errors as the separate calls; outputs untouched on error. */
ea_status ea_measure(ea_sim *sim, int slot, int r_max, int64_t *A, int64_t *B, int64_t *q, int64_t *E, int64_t *M);

/* Canonical packed I/O (host arrays: spins N words, bonds 3N words).
 * ea_set_bonds on a 2-replica sim: EA_ERR_INVALID unless hi half == lo half in every word (checked on the device
 * while packing: after this error the sim's bonds are undefined and must be set again). */
ea_status ea_get_spins(ea_sim *sim, uint64_t *host);
ea_status ea_set_spins(ea_sim *sim, const uint64_t *host);
ea_status ea_get_bonds(ea_sim *sim, uint64_t *host);
ea_status ea_set_bonds(ea_sim *sim, const uint64_t *host);
ea_status ea_get_snapshot(ea_sim *sim, int slot, uint64_t *host);

/* Batches: K independent small sims -- one L in {16, 32, 64}, one replica mode, 64 samples, one
 * device, one dynamics; each with its own p, T, seed and clock -- advanced by ONE kernel launch per colour for all of
 * them (such lattices are launch-bound alone).  ea_batch_sweep(b, n) is exactly ea_sweep(sim, n) on every member;
 * the members stay ordinary sims (observables, get/set, ea_sweep still work, correctly ordered across streams).
 * The batch runs on the first member's stream.  Destroy the batch before its members. */
typedef struct ea_batch ea_batch;
ea_status ea_batch_create(ea_sim *const *sims, int n_sims, ea_batch **out);
ea_status ea_batch_sweep(ea_batch *batch, uint64_t n);
ea_status ea_batch_destroy(ea_batch *batch);

/* Host-only self-test (no device needed): the tables of the RESIDENT kernel for both tile partitions (148 and 128 tiles) and
 * every number of compute warps -- the tiles cover the lattice exactly once, every row of a tile is scheduled exactly once in
 * its class with the boundary rows first, every halo row has an owner.  EA_OK or EA_ERR_STATE. */
ea_status ea_selftest_host(void);

/* Measured issue rates of the pipes that bound this library's kernels (the update is "boolean logic at
 * the bit level" plus one random number, and the observables are popcounts, Eq. 3 and 7): dependent-free
 * instruction streams on every SM of `device` (-1 = current), about 30 ms of device time, default stream.
 *   out[0] = LOP3 (alu pipe), out[1] = IMAD.WIDE.U32 (fma pipe), out[2] = POPC  -- warp instructions per second;
 *   out[3] = LOP3 rate while one IMAD.WIDE.U32 per four LOP3 is issued alongside (about the sweep kernel's mix).  Measured on
 *            B200: 4/5 of out[0] -- an IMAD.WIDE takes an alu-pipe issue slot besides its time on the fma pipe, so the
 *            alu roofline of the sweep kernel counts it as alu-pipe work;
 *   out[4] = SM clock in MHz during the LOP3 stream (clock64 / globaltimer), out[5] = number of SMs,
 *   out[6] = LOP3 rate while as many plain 32-bit IMAD are issued alongside (these do overlap), out[7] = 0.
 * host array of 8 doubles.  EA_ERR_CUDA without a device. */
ea_status ea_selftest_pipes(int device, double out[8]);

/* Philox4x32-10 block on the device (one thread), for the known-answer test of the GPU side (C-A6). */
ea_status ea_philox_selftest(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

const char *ea_strerror(ea_status s);
const char *ea_last_error(const ea_sim *sim);
const char *ea_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EA_B200_H */

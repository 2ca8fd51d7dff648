// ea_c4_vectors.cu -- the four-point correlation for arbitrary lattice vectors.
//
// Eq. 3: C_4(r, t_w) = (1/N) sum_i q_i q_{i+r}, "i + r ... a spin which has a spacial distance r
// from spin i" -- reading C-S8v: r is any lattice vector, periodic.  ea_c4 covers the axis vectors the paper fits
// (:112); this file covers the rest: the "all r >= 3" reference set (:112) and the merged points of Fig. 2.
//
// Layout.  The overlap field q_i = sigma^a_i ^ sigma^b_i (Eq. 2, one bit per disorder sample) is transposed once
// into x-rows:  Tr[((z L + y) WPR + w) 32 + b] = bits x = 32 w .. 32 w + 31 of row (y, z) of sample b
// (WPR = ceil(L / 32) words per row; N/32 x 32 words = 4 N bytes, kept in the staging buffer).
// A displacement (dx, dy, dz) is then: row (y + dy, z + dz), rotated right by dx bits inside the L-bit row;
// B_b(r) = N - 2 popcount over all rows of (row ^ shifted row).  Lane = sample, so every load is one 128-byte line.
//
// Work is cut into jobs = (dy, dz, first dx, up to NDX consecutive dx): the two rows are loaded once per job and
// the dx scan advances by one-bit funnel shifts.  The kernel is bound by the popcount rate (16 lanes / clk / SM).
#include <algorithm>
#include <mutex>
#include <vector>

#include "ea_internal.h"

namespace ea {

constexpr int C4V_NDX = 16;     // consecutive dx per job = popcount accumulators per thread
constexpr int C4V_ROWCHUNKS = 8; // CTAs per job along the rows

struct C4Job {
    int dy, dz, dx0, ndx; // dx0 already reduced to [0, L)
    unsigned out;         // first output slot (vector index in sorted order)
};

template <int WPR> struct RowWords { uint32_t w[WPR]; };

// rotate an L-bit row right by one bit (bit x of the result = bit x + 1 of the input, periodic)
template <int WPR>
__device__ __forceinline__ void rotr1(RowWords<WPR> &r, const int L)
{
    if (WPR == 1) {
        const uint32_t v = r.w[0];
        r.w[0] = L == 32 ? __funnelshift_r(v, v, 1) : ((v >> 1) | ((v & 1u) << (L - 1)));
    } else {
        const uint32_t first = r.w[0];
#pragma unroll
        for (int i = 0; i < WPR - 1; ++i) r.w[i] = __funnelshift_r(r.w[i], r.w[i + 1], 1);
        r.w[WPR - 1] = __funnelshift_r(r.w[WPR - 1], first, 1);
    }
}

// rotate right by d in [0, L)
template <int WPR>
__device__ __forceinline__ void rotr(RowWords<WPR> &r, const int L, int d)
{
    if (WPR == 1) {
        const uint32_t v = r.w[0];
        if (L == 32) r.w[0] = __funnelshift_r(v, v, d);
        else if (d) r.w[0] = ((v >> d) | (v << (L - d))) & (0xffffffffu >> (32 - L));
    } else {
        for (; d >= 32; d -= 32) { // whole words: uniform loop of register moves
            const uint32_t first = r.w[0];
#pragma unroll
            for (int i = 0; i < WPR - 1; ++i) r.w[i] = r.w[i + 1];
            r.w[WPR - 1] = first;
        }
        const uint32_t first = r.w[0];
#pragma unroll
        for (int i = 0; i < WPR - 1; ++i) r.w[i] = __funnelshift_r(r.w[i], r.w[i + 1], d);
        r.w[WPR - 1] = __funnelshift_r(r.w[WPR - 1], first, d);
    }
}

// spins (colour-split) -> Tr
__global__ void __launch_bounds__(256) k_q_rows(const Lattice lat, const uint64_t *__restrict__ spins, uint32_t *__restrict__ Tr,
                                                const int wpr)
{
    const unsigned lane = threadIdx.x & 31;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const unsigned L = lat.L, Lh = lat.Lh, n_items = L * L * wpr;
    for (unsigned it = warp; it < n_items; it += nwarps) { // warp-uniform
        const unsigned w = it % wpr, row = it / wpr, y = row % L, z = row / L;
        const unsigned x = 32 * w + lane;
        uint32_t q = 0;
        if (x < L) {
            const unsigned c = (x + y + z) & 1u;
            const uint64_t sg = spins[(size_t)c * lat.Nh + Lh * (y + L * z) + (x >> 1)];
            q = lo32(sg) ^ hi32(sg); // Eq. 2: q_i = S^a_i S^b_i  <->  sigma^a ^ sigma^b
        }
        Tr[(size_t)it * 32 + lane] = warp_transpose32(q, lane);
    }
}

template <int WPR>
__global__ void __launch_bounds__(256) k_c4_vec(const int L, const uint32_t *__restrict__ Tr, const C4Job *__restrict__ jobs,
                                                unsigned long long *__restrict__ out /* [n_vec][32] */)
{
    const C4Job job = jobs[blockIdx.y];
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    const unsigned n_rows = (unsigned)L * L;
    unsigned cnt[C4V_NDX];
#pragma unroll
    for (int i = 0; i < C4V_NDX; ++i) cnt[i] = 0;
    for (unsigned row = blockIdx.x * wpb + warp; row < n_rows; row += gridDim.x * wpb) {
        const unsigned y = row % L, z = row / L;
        unsigned y2 = y + job.dy, z2 = z + job.dz; // dy, dz already in [0, L)
        if (y2 >= (unsigned)L) y2 -= L;
        if (z2 >= (unsigned)L) z2 -= L;
        const unsigned row2 = z2 * L + y2;
        RowWords<WPR> a, b;
#pragma unroll
        for (int i = 0; i < WPR; ++i) {
            a.w[i] = __ldg(Tr + ((size_t)row * WPR + i) * 32 + lane);
            b.w[i] = __ldg(Tr + ((size_t)row2 * WPR + i) * 32 + lane);
        }
        rotr<WPR>(b, L, job.dx0);
#pragma unroll
        for (int i = 0; i < C4V_NDX; ++i) {
            if (i < job.ndx) { // uniform
                unsigned c = 0;
#pragma unroll
                for (int k = 0; k < WPR; ++k) c += __popc(a.w[k] ^ b.w[k]);
                cnt[i] += c;
                rotr1<WPR>(b, L);
            }
        }
    }
    __shared__ unsigned acc[C4V_NDX][32];
    for (unsigned k = threadIdx.x; k < C4V_NDX * 32; k += blockDim.x) (&acc[0][0])[k] = 0;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < C4V_NDX; ++i)
        if (i < job.ndx) atomicAdd(&acc[i][lane], cnt[i]);
    __syncthreads();
    for (unsigned k = threadIdx.x; k < (unsigned)job.ndx * 32; k += blockDim.x)
        atomicAdd(&out[(size_t)job.out * 32 + k], (unsigned long long)(&acc[0][0])[k]);
}

bool c4_vectors_supported(int L) { return L <= 32 || L == 64 || L == 128; }

// counts[v*32 + b] = number of sites with q_i != q_{i + r_v} for the n vectors (dx, dy, dz) in `vec` (any integers).
// Host result; synchronises the stream.
cudaError_t c4_vector_counts(ea_sim *s, size_t n, const int32_t *vec, unsigned long long *counts)
{
    const int L = s->lat.L;
    const int wpr = (L + 31) / 32;
    if (!n) return cudaSuccess;
    // sort by (dz, dy, dx) after reduction mod L, so that runs of consecutive dx share a job
    struct V { int dx, dy, dz; size_t idx; };
    std::vector<V> v(n);
    for (size_t i = 0; i < n; ++i) {
        auto m = [L](int a) { int r = a % L; return r < 0 ? r + L : r; };
        v[i] = {m(vec[3 * i]), m(vec[3 * i + 1]), m(vec[3 * i + 2]), i};
    }
    std::sort(v.begin(), v.end(), [](const V &a, const V &b) {
        if (a.dz != b.dz) return a.dz < b.dz;
        if (a.dy != b.dy) return a.dy < b.dy;
        if (a.dx != b.dx) return a.dx < b.dx;
        return a.idx < b.idx;
    });
    std::vector<C4Job> jobs;
    for (size_t i = 0; i < n;) {
        size_t j = i + 1;
        while (j < n && j - i < (size_t)C4V_NDX && v[j].dz == v[i].dz && v[j].dy == v[i].dy && v[j].dx == v[j - 1].dx + 1) ++j;
        jobs.push_back({v[i].dy, v[i].dz, v[i].dx, (int)(j - i), (unsigned)i});
        i = j;
    }
    // L^2 wpr 32 words of 4 B: fits the 8 N-byte staging buffer unless L < 16 (rows are padded to 32 bits)
    const size_t tr_bytes = (size_t)L * L * wpr * 32 * sizeof(uint32_t);
    uint32_t *Tr = (uint32_t *)s->stage, *Tr_own = nullptr;
    cudaError_t e;
    if (tr_bytes > (size_t)s->N * 8) {
        if ((e = cudaMalloc((void **)&Tr_own, tr_bytes)) != cudaSuccess) return e;
        Tr = Tr_own;
    }
    k_q_rows<<<(unsigned)s->n_sm * 2, 256, 0, s->stream>>>(s->lat, s->spins, Tr, wpr);
    s->count_launch();
    if ((e = cudaGetLastError()) != cudaSuccess) { if (Tr_own) cudaFree(Tr_own); return e; }

    const size_t JOBS_PER_PASS = 32768; // bounds the temporary buffers (grid.y <= 65535)
    std::vector<unsigned long long> h_out;
    auto grow = [](void **p, size_t *have, size_t need) -> cudaError_t { // the sim's grow-only scratch (freed by ea_destroy)
        if (*have >= need) return cudaSuccess;
        if (*p) cudaFree(*p);
        *p = nullptr;
        *have = 0;
        cudaError_t ge = cudaMalloc(p, need);
        if (ge == cudaSuccess) *have = need;
        return ge;
    };
    for (size_t j0 = 0; j0 < jobs.size(); j0 += JOBS_PER_PASS) {
        const size_t nj = std::min(JOBS_PER_PASS, jobs.size() - j0);
        const size_t v0 = jobs[j0].out, v1 = (j0 + nj < jobs.size()) ? jobs[j0 + nj].out : n;
        std::vector<C4Job> pass(jobs.begin() + j0, jobs.begin() + j0 + nj);
        for (auto &jb : pass) jb.out -= (unsigned)v0;
        if ((e = grow(&s->c4v_jobs, &s->c4v_jobs_bytes, nj * sizeof(C4Job))) != cudaSuccess) break;
        if ((e = grow((void **)&s->c4v_out, &s->c4v_out_bytes, (v1 - v0) * 32 * sizeof(unsigned long long))) != cudaSuccess) break;
        C4Job *d_jobs = (C4Job *)s->c4v_jobs;
        unsigned long long *d_out = s->c4v_out;
        if ((e = cudaMemcpyAsync(d_jobs, pass.data(), nj * sizeof(C4Job), cudaMemcpyHostToDevice, s->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(d_out, 0, (v1 - v0) * 32 * sizeof(unsigned long long), s->stream)) != cudaSuccess) break;
        const dim3 grid(C4V_ROWCHUNKS, (unsigned)nj);
        switch (wpr) {
        case 1: k_c4_vec<1><<<grid, 256, 0, s->stream>>>(L, Tr, d_jobs, d_out); break;
        case 2: k_c4_vec<2><<<grid, 256, 0, s->stream>>>(L, Tr, d_jobs, d_out); break;
        default: k_c4_vec<4><<<grid, 256, 0, s->stream>>>(L, Tr, d_jobs, d_out); break;
        }
        s->count_launch();
        if ((e = cudaGetLastError()) != cudaSuccess) break;
        h_out.resize((v1 - v0) * 32);
        if ((e = cudaMemcpyAsync(h_out.data(), d_out, h_out.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                                 s->stream)) != cudaSuccess) break;
        if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) break; // also keeps `pass` alive long enough
        for (size_t k = v0; k < v1; ++k)
            std::copy(h_out.begin() + (k - v0) * 32, h_out.begin() + (k - v0 + 1) * 32, counts + v[k].idx * 32);
    }
    if (Tr_own) { cudaStreamSynchronize(s->stream); cudaFree(Tr_own); }
    return e;
}

// ---------------------------------------------------------------------------------------------
// The same counts with NO device or host allocation (ea_c4_vectors_static, include/ea.h): for callers that cannot call
// cudaMalloc (inside a stream capture, in a serving loop, under a harness that forbids it).  c4_vector_counts() above keeps
// its job list and its counters in grow-only cudaMalloc buffers; here they live in ONE file-scope device array of a fixed,
// modest size, held by every GPU that loads the library until the process exits:
//     out    unsigned long long [C4V_STATIC_MAX_VECTORS][32]   256 KiB   counters, cleared at the start of every call
//     jobs   C4Job              [C4V_STATIC_MAX_VECTORS]        20 KiB
//     tr     uint32_t           [14 * 14 * 32]                  24.5 KiB  the transposed overlap field of an L < 16 lattice
//                                                                         (larger ones fit the sim's own staging buffer)
// In host code the array's NAME is only a host-side stand-in, not a device address: its address on a device comes from
// cudaGetSymbolAddress, asked once per device with that device current, below.  All calls share the array and it keeps
// the last call's contents: two calls that overlap on the GPU (two sims on two streams, two host threads) race.
// ---------------------------------------------------------------------------------------------
constexpr size_t C4V_STATIC_MAX_VECTORS = 1024; // = EA_C4_STATIC_MAX_VECTORS (include/ea.h; checked in ea_api.cu)
constexpr size_t C4V_STATIC_OUT_BYTES = C4V_STATIC_MAX_VECTORS * 32 * sizeof(unsigned long long);
constexpr size_t C4V_STATIC_JOBS_OFF = C4V_STATIC_OUT_BYTES;
constexpr size_t C4V_STATIC_JOBS_BYTES = (C4V_STATIC_MAX_VECTORS * sizeof(C4Job) + 255) / 256 * 256;
constexpr size_t C4V_STATIC_TR_OFF = C4V_STATIC_JOBS_OFF + C4V_STATIC_JOBS_BYTES;
constexpr size_t C4V_STATIC_TR_BYTES = (size_t)14 * 14 * 32 * sizeof(uint32_t);
constexpr size_t C4V_STATIC_BYTES = C4V_STATIC_TR_OFF + C4V_STATIC_TR_BYTES;

static __device__ __align__(256) unsigned char c4v_static_scratch[C4V_STATIC_BYTES];

constexpr int C4V_MAX_DEVICES = 64;
static unsigned char *c4v_static_ptr[C4V_MAX_DEVICES]; // device address of c4v_static_scratch, per device (nullptr: not asked yet)
static std::mutex c4v_static_mutex;

// the device address of the scratch array on `device`, which must be current
static cudaError_t c4v_static_address(int device, unsigned char **ptr)
{
    if (device < 0 || device >= C4V_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(c4v_static_mutex);
    if (!c4v_static_ptr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, c4v_static_scratch);
        if (e != cudaSuccess) return e;
        c4v_static_ptr[device] = (unsigned char *)p;
    }
    *ptr = c4v_static_ptr[device];
    return cudaSuccess;
}

size_t c4_vectors_static_max() { return C4V_STATIC_MAX_VECTORS; }

// As c4_vector_counts for n <= C4V_STATIC_MAX_VECTORS vectors (cudaErrorInvalidValue beyond): the same two kernels, scratch
// in the static array, host work in fixed-size buffers.  Synchronises the stream.  Not re-entrant (see above).
cudaError_t c4_vector_counts_static(ea_sim *s, size_t n, const int32_t *vec, unsigned long long *counts)
{
    if (n > C4V_STATIC_MAX_VECTORS) return cudaErrorInvalidValue;
    if (!n) return cudaSuccess;
    const int L = s->lat.L;
    const int wpr = (L + 31) / 32;
    unsigned char *scratch = nullptr;
    cudaError_t e = c4v_static_address(s->device, &scratch);
    if (e != cudaSuccess) return e;
    unsigned long long *d_out = (unsigned long long *)scratch;
    C4Job *d_jobs = (C4Job *)(scratch + C4V_STATIC_JOBS_OFF);

    // host side of c4_vector_counts in fixed-size buffers (static: 24 + 20 + 256 KiB are too much for a stack frame)
    struct V { int dx, dy, dz; unsigned idx; };
    static V v[C4V_STATIC_MAX_VECTORS];
    static C4Job jobs[C4V_STATIC_MAX_VECTORS];
    static unsigned long long h_out[C4V_STATIC_MAX_VECTORS * 32];
    static std::mutex host_mutex; // the host buffers; the DEVICE array is still shared by calls on other streams
    std::lock_guard<std::mutex> lock(host_mutex);
    for (size_t i = 0; i < n; ++i) {
        auto m = [L](int a) { int r = a % L; return r < 0 ? r + L : r; };
        v[i] = {m(vec[3 * i]), m(vec[3 * i + 1]), m(vec[3 * i + 2]), (unsigned)i};
    }
    std::sort(v, v + n, [](const V &a, const V &b) { // in place: no allocation
        if (a.dz != b.dz) return a.dz < b.dz;
        if (a.dy != b.dy) return a.dy < b.dy;
        if (a.dx != b.dx) return a.dx < b.dx;
        return a.idx < b.idx;
    });
    size_t nj = 0;
    for (size_t i = 0; i < n;) {
        size_t j = i + 1;
        while (j < n && j - i < (size_t)C4V_NDX && v[j].dz == v[i].dz && v[j].dy == v[i].dy && v[j].dx == v[j - 1].dx + 1) ++j;
        jobs[nj++] = {v[i].dy, v[i].dz, v[i].dx, (int)(j - i), (unsigned)i};
        i = j;
    }

    const size_t tr_bytes = (size_t)L * L * wpr * 32 * sizeof(uint32_t);
    uint32_t *Tr = (uint32_t *)s->stage;
    if (tr_bytes > (size_t)s->N * 8) { // L < 16 (rows are padded to 32 bits)
        if (tr_bytes > C4V_STATIC_TR_BYTES) return cudaErrorInvalidValue;
        Tr = (uint32_t *)(scratch + C4V_STATIC_TR_OFF);
    }
    k_q_rows<<<(unsigned)s->n_sm * 2, 256, 0, s->stream>>>(s->lat, s->spins, Tr, wpr);
    s->count_launch();
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(d_jobs, jobs, nj * sizeof(C4Job), cudaMemcpyHostToDevice, s->stream)) != cudaSuccess) return e;
    // the array keeps the last call's counters: the kernel adds into them, so they start at zero
    if ((e = cudaMemsetAsync(d_out, 0, n * 32 * sizeof(unsigned long long), s->stream)) != cudaSuccess) return e;
    const dim3 grid(C4V_ROWCHUNKS, (unsigned)nj);
    switch (wpr) {
    case 1: k_c4_vec<1><<<grid, 256, 0, s->stream>>>(L, Tr, d_jobs, d_out); break;
    case 2: k_c4_vec<2><<<grid, 256, 0, s->stream>>>(L, Tr, d_jobs, d_out); break;
    default: k_c4_vec<4><<<grid, 256, 0, s->stream>>>(L, Tr, d_jobs, d_out); break;
    }
    s->count_launch();
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(h_out, d_out, n * 32 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s->stream)) != cudaSuccess) return e;
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return e;
    for (size_t k = 0; k < n; ++k) std::copy(h_out + k * 32, h_out + (k + 1) * 32, counts + (size_t)v[k].idx * 32);
    return cudaSuccess;
}

} // namespace ea

// ea_observables.cu -- per-sample popcount reductions for the paper's observables (computed offline on a
// CPU in the paper): autocorrelation C(t,t_w) (Eq. 7, :63), replica overlap and C_4(r,t_w)
// along the lattice axes (Eq. 2-3, :31-40, :112), energy (Eq. 1, :23), magnetisation.
//
// Every observable is "N (or 3N) minus twice the number of set bits of sample b over a stream of words":
//   A_b = N - 2 cnt_b(sigma ^ sigma_snap),  M_b = N - 2 cnt_b(sigma),  E_b = -3N + 2 cnt_b(j ^ sigma_i ^ sigma_{i+e_d}),
//   B_b(d,r) = N - 2 cnt_b(Q_i ^ Q_{i + r e_d}),  Q_i = sigma^a_i ^ sigma^b_i,  q_b = N - 2 cnt_b(Q).
// A plain POPC counts across samples, so each warp first transposes its 32 words x 32 samples bit block
// (five shuffle butterflies), after which lane b holds 32 sites of sample b and POPC counts per sample.
#include "ea_internal.h"

namespace ea {

struct Coord { unsigned c, xh, y, z; };

__device__ __forceinline__ Coord coord_of(const Lattice &lat, unsigned e) // e in [0, N): (colour, compact index)
{
    Coord q;
    q.c = e >= lat.Nh;
    unsigned i = e - q.c * lat.Nh;
    q.xh = i % lat.Lh;
    unsigned row = i / lat.Lh;
    q.y = row % lat.L;
    q.z = row / lat.L;
    return q;
}

// flat index into spins[2][Nh] of canonical (x, y, z)
__device__ __forceinline__ unsigned flat_of(const Lattice &lat, unsigned x, unsigned y, unsigned z)
{
    unsigned c = (x + y + z) & 1u;
    return c * lat.Nh + (x >> 1) + lat.Lh * (y + lat.L * z);
}

// Accumulates, for this thread's lane b = threadIdx & 31, the set bits of samples b (lo) and b+32 (hi).
struct LaneCounter {
    unsigned lo = 0, hi = 0;
    __device__ __forceinline__ void add64(uint64_t w, unsigned lane)
    {
        lo += __popc(warp_transpose32(lo32(w), lane));
        hi += __popc(warp_transpose32(hi32(w), lane));
    }
    __device__ __forceinline__ void add32(uint32_t w, unsigned lane) { lo += __popc(warp_transpose32(w, lane)); }
};

// block reduce -> 64 (or 32) global counters
__device__ __forceinline__ void flush_counts(const LaneCounter &k, unsigned long long *out, bool both_halves)
{
    __shared__ unsigned acc[64];
    if (threadIdx.x < 64) acc[threadIdx.x] = 0;
    __syncthreads();
    unsigned lane = threadIdx.x & 31;
    atomicAdd(&acc[lane], k.lo);
    if (both_halves) atomicAdd(&acc[32 + lane], k.hi);
    __syncthreads();
    if (threadIdx.x < (both_halves ? 64 : 32)) atomicAdd(&out[threadIdx.x], (unsigned long long)acc[threadIdx.x]);
}

// cnt_b over all N words of sigma ^ other (other may be null): autocorrelation / magnetisation.
__global__ void __launch_bounds__(256) k_count_spins(Lattice lat, const uint64_t *__restrict__ spins,
                                                     const uint64_t *__restrict__ other, unsigned long long *out)
{
    const unsigned lane = threadIdx.x & 31, N = 2 * lat.Nh;
    const unsigned stride = gridDim.x * blockDim.x;
    LaneCounter k;
    for (unsigned base = blockIdx.x * blockDim.x; base < N; base += stride) { // block-uniform trip count
        unsigned e = base + threadIdx.x;
        uint64_t w = 0;
        if (e < N) w = other ? (spins[e] ^ other[e]) : spins[e];
        k.add64(w, lane);
    }
    flush_counts(k, out, true);
}

// cnt_b over the 3N words j_d(i) ^ sigma_i ^ sigma_{i+e_d} (unsatisfied bonds, C-A2): energy.
template <typename BondT>
__global__ void __launch_bounds__(256) k_count_energy(Lattice lat, const uint64_t *__restrict__ spins,
                                                      const BondT *__restrict__ bonds, unsigned long long *out)
{
    const unsigned lane = threadIdx.x & 31, N = 2 * lat.Nh;
    const unsigned stride = gridDim.x * blockDim.x;
    const unsigned L = lat.L, Lh = lat.Lh;
    LaneCounter k;
    for (unsigned base = blockIdx.x * blockDim.x; base < N; base += stride) {
        unsigned e = base + threadIdx.x;
        uint64_t u0 = 0, u1 = 0, u2 = 0;
        if (e < N) {
            Coord q = coord_of(lat, e);
            unsigned i = e - q.c * lat.Nh, x = 2 * q.xh + ((q.c ^ (q.y + q.z)) & 1u);
            unsigned xp = (x + 1 == L) ? 0 : x + 1, yp = (q.y + 1 == L) ? 0 : q.y + 1, zp = (q.z + 1 == L) ? 0 : q.z + 1;
            uint64_t sg = spins[e];
            const BondT *J = bonds + (size_t)q.c * 3 * lat.Nh;
            BondT j0 = J[i], j1 = J[lat.Nh + i], j2 = J[2 * lat.Nh + i];
            u0 = mk64(bond_lo(j0), bond_hi(j0)) ^ sg ^ spins[flat_of(lat, xp, q.y, q.z)];
            u1 = mk64(bond_lo(j1), bond_hi(j1)) ^ sg ^ spins[flat_of(lat, x, yp, q.z)];
            u2 = mk64(bond_lo(j2), bond_hi(j2)) ^ sg ^ spins[flat_of(lat, x, q.y, zp)];
            (void)Lh;
        }
        k.add64(u0, lane);
        k.add64(u1, lane);
        k.add64(u2, lane);
    }
    flush_counts(k, out, true);
}

// blockIdx.y = d*(r_max+1) + r for the displacement r e_d, or 3*(r_max+1) for the plain overlap.
__global__ void __launch_bounds__(256) k_count_c4(Lattice lat, const uint64_t *__restrict__ spins, int r_max,
                                                  unsigned long long *out)
{
    const unsigned lane = threadIdx.x & 31, N = 2 * lat.Nh, L = lat.L;
    const unsigned stride = gridDim.x * blockDim.x;
    const unsigned job = blockIdx.y, n_r = r_max + 1;
    const bool overlap_only = job == 3 * n_r;
    const unsigned d = overlap_only ? 0 : job / n_r, r = overlap_only ? 0 : job % n_r;
    LaneCounter k;
    for (unsigned base = blockIdx.x * blockDim.x; base < N; base += stride) {
        unsigned e = base + threadIdx.x;
        uint32_t w = 0;
        if (e < N) {
            uint64_t sg = spins[e];
            w = lo32(sg) ^ hi32(sg); // Q_i: bit 1 <-> q_i = S^a_i S^b_i = -1 (Eq. 2)
            if (!overlap_only) {
                Coord q = coord_of(lat, e);
                unsigned x = 2 * q.xh + ((q.c ^ (q.y + q.z)) & 1u), y = q.y, z = q.z;
                if (d == 0) { x += r; if (x >= L) x -= L; }
                if (d == 1) { y += r; if (y >= L) y -= L; }
                if (d == 2) { z += r; if (z >= L) z -= L; }
                uint64_t sn = spins[flat_of(lat, x, y, z)];
                w ^= lo32(sn) ^ hi32(sn);
            }
        }
        k.add32(w, lane);
    }
    flush_counts(k, out + (size_t)job * 32, false);
}

// ---------------------------------------------------------------------------------------------
// Fast C_4 path for L in {64, 128} (L/2 a multiple of 32), 2 replicas.
// Pass 1 (k_q_transpose): Q_i = sigma^a_i ^ sigma^b_i (Eq. 2), every block of 32 consecutive compact sites
// transposed once into sample-major words:  Tq[c][row][xb][b], row = y + L z, xb = block of 32 compact x
// positions; bit k of the word = Q of sample b at compact xh = 32 xb + k.  Also counts the overlap q.
// Pass 2: B_b(d, r) = N - 2 sum popc(own ^ partner): along y / z the partner of (c, row) at distance r is the
// word of colour c ^ (r & 1) in the row r further on (same xh: the row phase flips with the colour);
// along x it is the partner row's bits rotated by r/2 (r even, same colour) or (r-1)/2 + s (r odd, other
// colour, s = row phase of the own colour).  One POPC then counts 32 sites of one sample; lane = sample, so
// no cross-lane reduction is needed.
// ---------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(256) k_q_transpose(const uint64_t *__restrict__ spins, uint32_t *__restrict__ Tq,
                                                     unsigned long long *out_overlap)
{
    constexpr unsigned NW = (unsigned)L * L * L / 32; // 32-site blocks over both colours
    const unsigned lane = threadIdx.x & 31;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    unsigned cnt = 0;
    for (unsigned w = warp; w < NW; w += nwarps) { // warp-uniform trip count
        const uint64_t sg = spins[(size_t)w * 32 + lane];
        const uint32_t t = warp_transpose32(lo32(sg) ^ hi32(sg), lane);
        Tq[(size_t)w * 32 + lane] = t;
        cnt += __popc(t);
    }
    __shared__ unsigned acc[32];
    if (threadIdx.x < 32) acc[threadIdx.x] = 0;
    __syncthreads();
    atomicAdd(&acc[lane], cnt);
    __syncthreads();
    if (threadIdx.x < 32) atomicAdd(&out_overlap[threadIdx.x], (unsigned long long)acc[threadIdx.x]);
}

template <int NR>
__device__ __forceinline__ void flush_r_counts(const unsigned (&cnt)[NR], unsigned lane, int r_max,
                                               unsigned long long *out /* [r][32] */)
{
    __shared__ unsigned acc[NR][32];
    for (unsigned k = threadIdx.x; k < NR * 32; k += blockDim.x) (&acc[0][0])[k] = 0;
    __syncthreads();
#pragma unroll
    for (int r = 1; r < NR; ++r) atomicAdd(&acc[r][lane], cnt[r]);
    __syncthreads();
    for (unsigned k = threadIdx.x; k < NR * 32; k += blockDim.x)
        if ((int)(k >> 5) <= r_max && (&acc[0][0])[k]) atomicAdd(&out[k], (unsigned long long)(&acc[0][0])[k]);
}

// AXIS = 1 (y) or 2 (z)
template <int L, int AXIS>
__global__ void __launch_bounds__(256) k_c4_yz(const uint32_t *__restrict__ Tq, int r_max, unsigned long long *out)
{
    constexpr unsigned XB = L / 64, RW = XB * 32, PL = L * RW, CW = L * PL, NT = 2 * L * L * XB;
    constexpr int NR = L / 2 + 1;
    const unsigned lane = threadIdx.x & 31;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    unsigned cnt[NR];
#pragma unroll
    for (int r = 0; r < NR; ++r) cnt[r] = 0;
    for (unsigned t = warp; t < NT; t += nwarps) {
        const unsigned xb = t % XB, y = (t / XB) % L, z = (t / (XB * L)) % L, c = t / (XB * L * L);
        const uint32_t own = __ldg(Tq + c * CW + z * PL + y * RW + xb * 32 + lane);
#pragma unroll
        for (int r = 1; r < NR; ++r) {
            const unsigned cp = c ^ (r & 1);
            const unsigned yy = AXIS == 1 ? ((y + r) & (L - 1)) : y, zz = AXIS == 2 ? ((z + r) & (L - 1)) : z;
            cnt[r] += __popc(own ^ __ldg(Tq + cp * CW + zz * PL + yy * RW + xb * 32 + lane));
        }
    }
    flush_r_counts<NR>(cnt, lane, r_max, out);
}

template <int L> struct RowBits;
template <> struct RowBits<128> {
    typedef uint64_t type;
    static __device__ __forceinline__ uint64_t load(const uint32_t *p) { return mk64(__ldg(p), __ldg(p + 32)); }
    static __device__ __forceinline__ uint64_t rotr(uint64_t v, unsigned d) { return (v >> d) | (v << ((64 - d) & 63)); }
    static __device__ __forceinline__ unsigned popc(uint64_t v) { return __popcll(v); }
};
template <> struct RowBits<64> {
    typedef uint32_t type;
    static __device__ __forceinline__ uint32_t load(const uint32_t *p) { return __ldg(p); }
    static __device__ __forceinline__ uint32_t rotr(uint32_t v, unsigned d) { return (v >> d) | (v << ((32 - d) & 31)); }
    static __device__ __forceinline__ unsigned popc(uint32_t v) { return __popc(v); }
};

template <int L>
__global__ void __launch_bounds__(256) k_c4_x(const uint32_t *__restrict__ Tq, int r_max, unsigned long long *out)
{
    constexpr unsigned XB = L / 64, RW = XB * 32, CW = (unsigned)L * L * RW, NT = L * L;
    constexpr int NR = L / 2 + 1;
    typedef RowBits<L> RB;
    const unsigned lane = threadIdx.x & 31;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    unsigned cnt[NR];
#pragma unroll
    for (int r = 0; r < NR; ++r) cnt[r] = 0;
    for (unsigned row = warp; row < NT; row += nwarps) {
        const unsigned y = row % L, z = row / L, s0 = (y + z) & 1u; // row phase of colour 0; colour 1 has 1 - s0
        const typename RB::type R0 = RB::load(Tq + row * RW + lane), R1 = RB::load(Tq + CW + row * RW + lane);
#pragma unroll
        for (int r = 1; r < NR; ++r) {
            const unsigned e = r >> 1;
            if ((r & 1) == 0)
                cnt[r] += RB::popc(R0 ^ RB::rotr(R0, e)) + RB::popc(R1 ^ RB::rotr(R1, e));
            else
                cnt[r] += RB::popc(R0 ^ RB::rotr(R1, e + s0)) + RB::popc(R1 ^ RB::rotr(R0, e + 1 - s0));
        }
    }
    flush_r_counts<NR>(cnt, lane, r_max, out);
}

template <int L>
static cudaError_t launch_c4_fast(ea_sim *s, int r_max)
{
    const size_t n_r = (size_t)r_max + 1;
    uint32_t *Tq = (uint32_t *)s->stage; // N words of 4 B in the 8 N-byte canonical staging buffer
    const unsigned grid = (unsigned)s->n_sm * 2;
    k_q_transpose<L><<<grid, 256, 0, s->stream>>>(s->spins, Tq, s->counters + 3 * n_r * 32);
    s->count_launch();
    k_c4_x<L><<<grid, 256, 0, s->stream>>>(Tq, r_max, s->counters);
    s->count_launch();
    k_c4_yz<L, 1><<<grid, 256, 0, s->stream>>>(Tq, r_max, s->counters + n_r * 32);
    s->count_launch();
    k_c4_yz<L, 2><<<grid, 256, 0, s->stream>>>(Tq, r_max, s->counters + 2 * n_r * 32);
    return cudaGetLastError();
}

static unsigned grid_for(const ea_sim *s, size_t items)
{
    size_t need = (items + 255) / 256, cap = (size_t)s->n_sm * 8;
    return (unsigned)(need < cap ? (need ? need : 1) : cap);
}

cudaError_t launch_count_spins(ea_sim *s, const uint64_t *d_other)
{
    cudaError_t e = cudaMemsetAsync(s->counters, 0, 64 * sizeof(unsigned long long), s->stream);
    if (e != cudaSuccess) return e;
    k_count_spins<<<grid_for(s, s->N), 256, 0, s->stream>>>(s->lat, s->spins, d_other, s->counters);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_count_energy(ea_sim *s)
{
    cudaError_t e = cudaMemsetAsync(s->counters, 0, 64 * sizeof(unsigned long long), s->stream);
    if (e != cudaSuccess) return e;
    if (s->n_replicas == 2)
        k_count_energy<uint32_t><<<grid_for(s, s->N), 256, 0, s->stream>>>(s->lat, s->spins, (const uint32_t *)s->bonds, s->counters);
    else
        k_count_energy<uint64_t><<<grid_for(s, s->N), 256, 0, s->stream>>>(s->lat, s->spins, (const uint64_t *)s->bonds, s->counters);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_count_c4(ea_sim *s, int r_max)
{
    size_t jobs = 3 * (size_t)(r_max + 1) + 1;
    cudaError_t e = cudaMemsetAsync(s->counters, 0, jobs * 32 * sizeof(unsigned long long), s->stream);
    if (e != cudaSuccess) return e;
    if (s->lat.L == 128 || s->lat.L == 64) { // r = 0 is B = N exactly: its counters stay 0
        e = s->lat.L == 128 ? launch_c4_fast<128>(s, r_max) : launch_c4_fast<64>(s, r_max);
        s->count_launch();
        return e;
    }
    size_t need = ((size_t)s->N + 255) / 256, cap = (size_t)s->n_sm * 2;
    dim3 grid((unsigned)(need < cap ? need : cap), (unsigned)jobs);
    k_count_c4<<<grid, 256, 0, s->stream>>>(s->lat, s->spins, r_max, s->counters);
    s->count_launch();
    return cudaGetLastError();
}

} // namespace ea

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

// block reduce -> 64 (or 32) global counters.  After the warp-shuffle transposition a lane holds the counts of ITS two samples
// (lane, lane + 32), so nothing is left to reduce across lanes; the warps of the CTA are summed through shared memory
// (one slot per warp and sample, no atomics) and one thread per sample adds the CTA's total to the global counter.
__device__ __forceinline__ void flush_counts(const LaneCounter &k, unsigned long long *out, bool both_halves)
{
    __shared__ unsigned acc[8][64]; // launch bounds: 256 threads
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    acc[warp][lane] = k.lo;
    acc[warp][32 + lane] = k.hi;
    __syncthreads();
    if (threadIdx.x < (both_halves ? 64u : 32u)) {
        unsigned long long t = 0;
        for (unsigned w = 0; w < nw; ++w) t += acc[w][threadIdx.x];
        if (t) atomicAdd(&out[threadIdx.x], t);
    }
}

// Bit-sliced (vertical) per-sample counter.  Eight 64-sample words go through seven 3:2 compressors (Harley-Seal) into
// ones / twos / fours planes kept per thread; the "eights" word they emit ripples through four more planes (weights 8 ..
// 64) with half adders, so that nothing pays for the 32 x 32 bit transposition and the POPC until a thread has taken 120
// words (or is done): seven planes are drained at once instead of one transposition per eight words.
struct VCounter {
    uint64_t ones = 0, twos = 0, fours = 0, hi[4] = {0, 0, 0, 0}; // hi[k]: weight 8 << k
    unsigned n_words = 0;                                         // taken since the last drain (thread-uniform in a warp)
    static __device__ __forceinline__ void csa(uint64_t &h, uint64_t &l, uint64_t a, uint64_t b, uint64_t c)
    {
        h = mk64(lop3<LUT_MAJ>(lo32(a), lo32(b), lo32(c)), lop3<LUT_MAJ>(hi32(a), hi32(b), hi32(c)));
        l = mk64(lop3<LUT_XOR3>(lo32(a), lo32(b), lo32(c)), lop3<LUT_XOR3>(hi32(a), hi32(b), hi32(c)));
    }
    // weights x planes -> counts of the lane's two samples; planes cleared
    __device__ __forceinline__ void drain(LaneCounter &k, unsigned lane)
    {
        LaneCounter t;
        unsigned lo = 0, hi_ = 0;
#pragma unroll
        for (int l = 3; l >= 0; --l) {
            t.lo = t.hi = 0;
            t.add64(hi[l], lane);
            lo = 2 * lo + t.lo;
            hi_ = 2 * hi_ + t.hi;
            hi[l] = 0;
        }
        const uint64_t low[3] = {fours, twos, ones};
#pragma unroll
        for (int l = 0; l < 3; ++l) {
            t.lo = t.hi = 0;
            t.add64(low[l], lane);
            lo = 2 * lo + t.lo;
            hi_ = 2 * hi_ + t.hi;
        }
        ones = twos = fours = 0;
        n_words = 0;
        k.lo += lo;
        k.hi += hi_;
    }
    __device__ __forceinline__ void add8(const uint64_t (&x)[8], LaneCounter &k, unsigned lane)
    {
        if (n_words > 127 - 8) drain(k, lane); // the planes hold counts up to 127
        uint64_t tA, tB, tC, tD, fA, fB, e;
        csa(tA, ones, ones, x[0], x[1]);
        csa(tB, ones, ones, x[2], x[3]);
        csa(fA, twos, twos, tA, tB);
        csa(tC, ones, ones, x[4], x[5]);
        csa(tD, ones, ones, x[6], x[7]);
        csa(fB, twos, twos, tC, tD);
        csa(e, fours, fours, fA, fB);
#pragma unroll
        for (int l = 0; l < 4; ++l) { // half adders: the carry out of the last plane is zero by the bound above
            const uint64_t c = hi[l] & e;
            hi[l] ^= e;
            e = c;
        }
        n_words += 8;
    }
};

// cnt_b over all N words of sigma ^ other (other may be null): autocorrelation / magnetisation.
__global__ void __launch_bounds__(256) k_count_spins(Lattice lat, const uint64_t *__restrict__ spins,
                                                     const uint64_t *__restrict__ other, unsigned long long *out)
{
    const unsigned lane = threadIdx.x & 31, N = 2 * lat.Nh;
    const unsigned stride = gridDim.x * blockDim.x;
    VCounter acc;
    LaneCounter k;
    for (unsigned base = blockIdx.x * blockDim.x; base < N; base += 8 * stride) { // block-uniform trip count
        uint64_t w[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const unsigned e = base + j * stride + threadIdx.x;
            w[j] = e < N ? (other ? (spins[e] ^ other[e]) : spins[e]) : 0;
        }
        acc.add8(w, k, lane);
    }
    acc.drain(k, lane);
    flush_counts(k, out, true);
}

// cnt_b over the 3N words j_d(i) ^ sigma_i ^ sigma_{i+e_d} (unsatisfied bonds, C-A2): energy.
// POW2: L is a power of two -- coordinates by shifts and masks (the divisions by run-time L cost more than the counting)
template <typename BondT, bool POW2>
__global__ void __launch_bounds__(256) k_count_energy(Lattice lat, const uint64_t *__restrict__ spins,
                                                      const BondT *__restrict__ bonds, unsigned long long *out)
{
    const unsigned lane = threadIdx.x & 31, Nh = lat.Nh, N = 2 * Nh;
    const unsigned stride = gridDim.x * blockDim.x;
    const unsigned L = lat.L, Lh = lat.Lh;
    VCounter acc;
    LaneCounter k;
    for (unsigned base = blockIdx.x * blockDim.x; base < N; base += 8 * stride) { // eight sites = three groups of eight words
        uint64_t u[3][8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const unsigned e = base + j * stride + threadIdx.x;
            u[0][j] = u[1][j] = u[2][j] = 0;
            if (e < N) {
                const unsigned c = e >= Nh, i = e - c * Nh;
                unsigned xh, y, z;
                if (POW2) {
                    xh = i & (Lh - 1);
                    const unsigned row = i >> lat.log2Lh;
                    y = row & (L - 1);
                    z = row >> lat.log2L;
                } else {
                    xh = i % Lh;
                    const unsigned row = i / Lh;
                    y = row % L;
                    z = row / L;
                }
                // the +x / +y / +z neighbours have the other colour: compact x = xh + S (S = row phase of colour c), same xh
                const unsigned S = (c ^ (y + z)) & 1u, xn = xh + S == Lh ? 0 : xh + S;
                const unsigned yp = y + 1 == L ? 0 : y + 1, zp = z + 1 == L ? 0 : z + 1;
                const uint64_t *oth = spins + (1 - c) * Nh;
                const uint64_t sg = spins[e];
                const BondT *J = bonds + (size_t)c * 3 * Nh;
                const BondT j0 = J[i], j1 = J[Nh + i], j2 = J[2 * Nh + i];
                u[0][j] = mk64(bond_lo(j0), bond_hi(j0)) ^ sg ^ oth[i - xh + xn];
                u[1][j] = mk64(bond_lo(j1), bond_hi(j1)) ^ sg ^ oth[Lh * (yp + L * z) + xh];
                u[2][j] = mk64(bond_lo(j2), bond_hi(j2)) ^ sg ^ oth[Lh * (y + L * zp) + xh];
            }
        }
#pragma unroll
        for (int d = 0; d < 3; ++d) acc.add8(u[d], k, lane);
    }
    acc.drain(k, lane);
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
    for (unsigned w0 = warp; w0 < NW; w0 += 4 * nwarps) { // warp-uniform trip count; four loads in flight
        uint64_t sg[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const unsigned w = w0 + j * nwarps;
            sg[j] = w < NW ? spins[(size_t)w * 32 + lane] : 0;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const unsigned w = w0 + j * nwarps;
            if (w < NW) {
                const uint32_t t = warp_transpose32(lo32(sg[j]) ^ hi32(sg[j]), lane);
                Tq[(size_t)w * 32 + lane] = t;
                cnt += __popc(t);
            }
        }
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

// AXIS = 1 (y) or 2 (z).  One CTA of four warps stages one COLUMN of the transposed field -- the L rows along the axis
// at fixed (z or y, xb), both colours, 32 KB, by cp.async -- in shared memory and handles 16 of the L/2 distances: a warp
// takes eight distances and the own rows of one colour.
// For a block of eight rows the own words stay in registers while each distance streams its eight partner rows in
// (rows L .. L+7 repeat rows 0 .. 7, so a block never wraps); the eight XOR words of a (block, distance) go through a
// carry-save adder tree (Harley-Seal: seven 3:2 compressors = 14 LOP3) into bit-sliced ones / twos / fours planes per
// distance, and only the "eights" word is popcounted: one POPC per eight site words instead of eight, which moves the
// kernel from the POPC rate (one warp instruction per 8 clocks) to the LOP3 rate.
template <int L, int AXIS>
__global__ void __launch_bounds__(128) k_c4_yz(const uint32_t *__restrict__ Tq, int r_max, unsigned long long *out)
{
    constexpr unsigned XB = L / 64, RW = XB * 32, PL = L * RW, CW = L * PL;
    constexpr int NR = L / 2, RPW = 8, RPC = 16, NCHUNK = NR / RPC, BLK = 8;
    static_assert(NR % RPC == 0 && L % BLK == 0, "distances and rows come in whole blocks");
    __shared__ __align__(16) uint32_t col[2][L + BLK][32];
    const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned chunk = blockIdx.x % NCHUNK, colid = blockIdx.x / NCHUNK;
    const unsigned xb = colid % XB, u = colid / XB; // u = z (AXIS 1) or y (AXIS 2)
    // a row of the column is 128 contiguous bytes of Tq: eight threads x 16 bytes
    for (unsigned i = tid; i < 2u * (L + BLK) * 8; i += 128) {
        const unsigned q = i & 7, rowx = (i >> 3) % (L + BLK), c = (i >> 3) / (L + BLK), row = rowx & (L - 1);
        const unsigned idx = (AXIS == 1 ? c * CW + u * PL + row * RW : c * CW + row * PL + u * RW) + xb * 32 + 4 * q;
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&col[c][rowx][4 * q]);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(Tq + idx) : "memory");
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    const unsigned c = warp & 1; // colour of the own rows
    const unsigned r0 = 1 + chunk * RPC + (warp >> 1) * RPW; // odd: distance r0 + ri flips the colour iff ri is even
    uint32_t ones[RPW], twos[RPW], fours[RPW], cnt[RPW];
#pragma unroll
    for (int ri = 0; ri < RPW; ++ri) ones[ri] = twos[ri] = fours[ri] = cnt[ri] = 0;
#pragma unroll 1
    for (unsigned y0 = 0; y0 < (unsigned)L; y0 += BLK) {
            uint32_t own[BLK];
#pragma unroll
            for (int j = 0; j < BLK; ++j) own[j] = col[c][y0 + j][lane];
#pragma unroll
            for (int ri = 0; ri < RPW; ++ri) {
                const uint32_t *pr = &col[c ^ ((1 + ri) & 1)][(y0 + r0 + ri) & (L - 1)][lane];
                uint32_t x[BLK];
#pragma unroll
                for (int j = 0; j < BLK; ++j) x[j] = own[j] ^ pr[j * 32];
                // carry-save: (ones, x0, x1) -> ones, twosA; ... ; (fours, foursA, foursB) -> fours, eights
                const uint32_t tA = lop3<LUT_MAJ>(ones[ri], x[0], x[1]), o1 = lop3<LUT_XOR3>(ones[ri], x[0], x[1]);
                const uint32_t tB = lop3<LUT_MAJ>(o1, x[2], x[3]), o2 = lop3<LUT_XOR3>(o1, x[2], x[3]);
                const uint32_t fA = lop3<LUT_MAJ>(twos[ri], tA, tB), t1 = lop3<LUT_XOR3>(twos[ri], tA, tB);
                const uint32_t tC = lop3<LUT_MAJ>(o2, x[4], x[5]), o3 = lop3<LUT_XOR3>(o2, x[4], x[5]);
                const uint32_t tD = lop3<LUT_MAJ>(o3, x[6], x[7]), o4 = lop3<LUT_XOR3>(o3, x[6], x[7]);
                const uint32_t fB = lop3<LUT_MAJ>(t1, tC, tD), t2 = lop3<LUT_XOR3>(t1, tC, tD);
                const uint32_t e = lop3<LUT_MAJ>(fours[ri], fA, fB);
                fours[ri] = lop3<LUT_XOR3>(fours[ri], fA, fB);
                ones[ri] = o4;
                twos[ri] = t2;
                cnt[ri] += __popc(e);
            }
        }
#pragma unroll
    for (int ri = 0; ri < RPW; ++ri) {
        const unsigned r = r0 + ri;
        const unsigned total = 8 * cnt[ri] + 4 * __popc(fours[ri]) + 2 * __popc(twos[ri]) + __popc(ones[ri]);
        if ((int)r <= r_max && total) atomicAdd(&out[r * 32 + lane], (unsigned long long)total);
    }
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
    constexpr unsigned grid_yz = (unsigned)L * (L / 64) * ((L / 2) / 16); // columns x chunks of 16 distances
    k_c4_yz<L, 1><<<grid_yz, 128, 0, s->stream>>>(Tq, r_max, s->counters + n_r * 32);
    s->count_launch();
    k_c4_yz<L, 2><<<grid_yz, 128, 0, s->stream>>>(Tq, r_max, s->counters + 2 * n_r * 32);
    return cudaGetLastError();
}

// Counting kernels: every thread ends with the transposition of its seven planes, so threads are few and long -- two
// CTAs of 256 threads per SM (L = 128: 28 words per thread) unless the lattice has fewer words than that
static unsigned grid_for(const ea_sim *s, size_t items)
{
    size_t need = (items + 255) / 256, cap = (size_t)s->n_sm * 2;
    return (unsigned)(need < cap ? (need ? need : 1) : cap);
}

cudaError_t launch_count_spins(ea_sim *s, const uint64_t *d_other, unsigned long long *dst)
{
    if (!dst) dst = s->counters;
    cudaError_t e = cudaMemsetAsync(dst, 0, 64 * sizeof(unsigned long long), s->stream);
    if (e != cudaSuccess) return e;
    k_count_spins<<<grid_for(s, s->N), 256, 0, s->stream>>>(s->lat, s->spins, d_other, dst);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_count_energy(ea_sim *s, unsigned long long *dst)
{
    if (!dst) dst = s->counters;
    cudaError_t e = cudaMemsetAsync(dst, 0, 64 * sizeof(unsigned long long), s->stream);
    if (e != cudaSuccess) return e;
    const bool pow2 = s->lat.log2L >= 0 && s->lat.log2Lh >= 0;
    const unsigned grid = grid_for(s, s->N);
    if (s->n_replicas == 2) {
        if (pow2) k_count_energy<uint32_t, true><<<grid, 256, 0, s->stream>>>(s->lat, s->spins, (const uint32_t *)s->bonds, dst);
        else k_count_energy<uint32_t, false><<<grid, 256, 0, s->stream>>>(s->lat, s->spins, (const uint32_t *)s->bonds, dst);
    } else {
        if (pow2) k_count_energy<uint64_t, true><<<grid, 256, 0, s->stream>>>(s->lat, s->spins, (const uint64_t *)s->bonds, dst);
        else k_count_energy<uint64_t, false><<<grid, 256, 0, s->stream>>>(s->lat, s->spins, (const uint64_t *)s->bonds, dst);
    }
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

// ea_fold.cu -- mixed multispin coding with M < 64 samples per word (III).  The paper's
// recipe, restated: with M = 2^m < 64 samples, a word carries 64/M sites of every sample -- the lattice is cut into 64/M
// equal parts along one dimension and the sites at the same relative position of each part share a word (bits i, i + M,
// i + 2M, ... belong to sample i).  The sweep then runs on a lattice 64/M times smaller, except across the cut, where the
// neighbouring word has to be rotated by M bits.
//
// Here: K = 64/M slabs along z, folded lattice L x L x Lz (Lz = L/K, even so that folded and physical colour agree);
// bit j + M k of folded word (x, y, z') = sample j at physical site (x, y, z' + k Lz).  The +z neighbour of the top
// plane z' = Lz - 1 is plane z' = 0 rotated right by M (slab k sees slab k + 1; the last slab wraps to the first);
// the -z neighbour of z' = 0 is plane Lz - 1 rotated left by M, and so is its bond word.
//
// Contract (DESIGN.md C-M): the M samples ARE samples of the 64-sample definition -- sample j is standard lane
// lam(j) (2 replicas: j < M/2 -> lane j = disorder j replica (a), else lane 32 + j - M/2 = the same disorder's
// replica (b); 1 replica: lane j) -- with the same bonds, the same start and the same random numbers, which are
// keyed by the PHYSICAL site: every word needs 2 K numbers (the paper's "64/M random numbers", :94).  A folded sim
// is therefore bit-identical to the used lanes of the 64-sample sim of the same seed, and the oracle needs no
// folded mode at all.
//
// The standard (unfolded) layout stays the exchange format inside the library: setup, get/set and every observable
// kernel work on it; k_fold / k_unfold convert.  Only the sweep runs on folded words.
#include "ea_internal.h"

namespace ea {

struct FoldGeom {
    int M, K;          // samples per word, slabs
    int n_replicas;
    unsigned Nhf;      // folded words per colour = Nh / K
    unsigned Lz;       // folded planes = L / K
    uint64_t g_lo;     // group bits whose sample uses the first random number of its site (standard lanes 0..31)
    uint64_t g_hi;     // ... the second (standard lanes 32..63)
};

static FoldGeom fold_geom(const ea_sim *s)
{
    FoldGeom f;
    f.M = s->n_samples;
    f.K = 64 / f.M;
    f.n_replicas = s->n_replicas;
    f.Nhf = s->lat.Nh / f.K;
    f.Lz = s->lat.L / f.K;
    if (s->n_replicas == 2) {
        f.g_lo = ((uint64_t)1 << (f.M / 2)) - 1;
        f.g_hi = f.g_lo << (f.M / 2);
    } else {
        f.g_lo = f.M == 64 ? ~(uint64_t)0 : ((uint64_t)1 << f.M) - 1; // M <= 32 independent samples: lanes 0..M-1
        f.g_hi = 0;
    }
    return f;
}

// standard 64-lane word -> the M group bits (C-M)
__device__ __forceinline__ uint64_t compress_lanes(const FoldGeom &f, uint64_t w)
{
    if (f.n_replicas == 2) return (w & f.g_lo) | (((w >> 32) & f.g_lo) << (f.M / 2));
    return w & f.g_lo;
}
__device__ __forceinline__ uint64_t expand_lanes(const FoldGeom &f, uint64_t g)
{
    if (f.n_replicas == 2) return (g & f.g_lo) | (((g >> (f.M / 2)) & f.g_lo) << 32);
    return g & f.g_lo;
}

// standard spins [2][Nh] -> folded [2][Nhf]
__global__ void k_fold_spins(const FoldGeom f, const unsigned Nh, const uint64_t *__restrict__ std_, uint64_t *__restrict__ fold)
{
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * f.Nhf) return;
    const unsigned c = tid >= f.Nhf, i = tid - c * f.Nhf;
    uint64_t w = 0;
    for (int k = 0; k < f.K; ++k) w |= compress_lanes(f, std_[(size_t)c * Nh + i + (size_t)k * f.Nhf]) << (f.M * k);
    fold[tid] = w;
}

// folded spins -> standard (unused lanes zero)
__global__ void k_unfold_spins(const FoldGeom f, const unsigned Nh, const uint64_t *__restrict__ fold, uint64_t *__restrict__ std_)
{
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * f.Nhf) return;
    const unsigned c = tid >= f.Nhf, i = tid - c * f.Nhf;
    const uint64_t w = fold[tid];
    for (int k = 0; k < f.K; ++k) std_[(size_t)c * Nh + i + (size_t)k * f.Nhf] = expand_lanes(f, w >> (f.M * k));
}

// standard bonds BondT [2][3][Nh] -> folded uint64 [2][3][Nhf]; 2 replicas: both replicas get the disorder's bit
template <typename BondT>
__global__ void k_fold_bonds(const FoldGeom f, const unsigned Nh, const BondT *__restrict__ std_, uint64_t *__restrict__ fold)
{
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 6 * f.Nhf) return;
    const unsigned plane = tid / f.Nhf, i = tid - plane * f.Nhf; // plane = c * 3 + d
    uint64_t w = 0;
    for (int k = 0; k < f.K; ++k) {
        const uint64_t b = (uint64_t)std_[(size_t)plane * Nh + i + (size_t)k * f.Nhf];
        const uint64_t g = f.n_replicas == 2 ? ((b & f.g_lo) | ((b & f.g_lo) << (f.M / 2))) : (b & f.g_lo);
        w |= g << (f.M * k);
    }
    fold[tid] = w;
}

template <typename T> __global__ void k_mask_words(T *p, size_t n, T mask)
{
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid < n) p[tid] &= mask;
}

__device__ __forceinline__ uint64_t rotr64(uint64_t v, int d) { return (v >> d) | (v << ((64 - d) & 63)); }
__device__ __forceinline__ uint64_t rotl64(uint64_t v, int d) { return (v << d) | (v >> ((64 - d) & 63)); }

struct FoldSweepArgs {
    FoldGeom f;
    Lattice lat;
    int colour;
    uint64_t *own;        // folded spins[colour]
    const uint64_t *oth;  // folded spins[1 - colour]
    const uint64_t *Jc;   // folded bonds[colour][3][Nhf]
    const uint64_t *Jo;   // folded bonds[1 - colour][3][Nhf]
    uint64_t seed, t;
    const uint64_t *d_time;
    uint32_t t_offset;
    Thresholds th;        // 32-bit thresholds + "always" flags (thr == 2^32, T = inf)
};

// flip word of one 64-bit multispin given the level masks m_k (bit set <=> that sample's number is below thr[k])
__device__ __forceinline__ uint64_t flip_word_masks(uint64_t s, uint64_t n1, uint64_t n2, uint64_t n3, uint64_t n4, uint64_t n5,
                                                    uint64_t n6, uint64_t j1, uint64_t j2, uint64_t j3, uint64_t j4, uint64_t j5,
                                                    uint64_t j6, uint64_t m0, uint64_t m1, uint64_t m2)
{
    const uint64_t u1 = j1 ^ s ^ n1, u2 = j2 ^ s ^ n2, u3 = j3 ^ s ^ n3, u4 = j4 ^ s ^ n4, u5 = j5 ^ s ^ n5, u6 = j6 ^ s ^ n6;
    const uint64_t sa = u1 ^ u2 ^ u3, ka = (u1 & u2) | (u3 & (u1 | u2));
    const uint64_t sb = u4 ^ u5 ^ u6, kb = (u4 & u5) | (u6 & (u4 | u5));
    const uint64_t t = sa | sb;
    uint64_t f = (ka & kb) | (t & (ka | kb)); // [n_u >= 3]: Delta E <= 0, always flipped
    if (m2) {                                 // some sample of this word drew a number below thr[2] (rare at low T)
        const uint64_t ge2 = ka | kb | (sa & sb), ge1 = ka | kb | t;
        f |= (m2 & ge2) | (m1 & ge1) | m0;    // Eq. 9 with nested thresholds (see flip_half): m0 <= m1 <= m2 bitwise
    }
    return f;
}

// Heat bath (reading C-HB): flip with probability hb[n_u], n_u = 0..6 unsatisfied bonds, hb increasing in n_u.  With the
// level masks m_k (bit set <=> that sample's number is below hb[k], nested: m_0 <= ... <= m_6 bitwise) the flip word is
// m_{n_u} = OR_k (m_k & [n_u >= k]); n_u = d0 + 2 d1 + 4 d2 from the two full adders.
__device__ __forceinline__ uint64_t flip_word_masks_heatbath(uint64_t s, uint64_t n1, uint64_t n2, uint64_t n3, uint64_t n4,
                                                             uint64_t n5, uint64_t n6, uint64_t j1, uint64_t j2, uint64_t j3,
                                                             uint64_t j4, uint64_t j5, uint64_t j6, const uint64_t (&m)[7])
{
    const uint64_t u1 = j1 ^ s ^ n1, u2 = j2 ^ s ^ n2, u3 = j3 ^ s ^ n3, u4 = j4 ^ s ^ n4, u5 = j5 ^ s ^ n5, u6 = j6 ^ s ^ n6;
    const uint64_t sa = u1 ^ u2 ^ u3, ka = (u1 & u2) | (u3 & (u1 | u2));
    const uint64_t sb = u4 ^ u5 ^ u6, kb = (u4 & u5) | (u6 & (u4 | u5));
    const uint64_t d0 = sa ^ sb, c0 = sa & sb;
    const uint64_t d1 = ka ^ kb ^ c0, d2 = (ka & kb) | (c0 & (ka | kb));
    const uint64_t ge1 = d0 | d1 | d2, ge2 = d1 | d2, ge3 = d2 | (d1 & d0), ge4 = d2, ge5 = d2 & (d1 | d0), ge6 = d2 & d1;
    return m[0] | (m[1] & ge1) | (m[2] & ge2) | (m[3] & ge3) | (m[4] & ge4) | (m[5] & ge5) | (m[6] & ge6);
}

// one thread = two x-adjacent folded words of one colour (L % 4 == 0)
// MT = M as a compile-time constant (shifts and the slab loop unroll), or 0: taken from the arguments.
// POW2: L is a power of two (index arithmetic by shifts).
template <int MT, bool POW2, bool ALWAYS, bool HB = false>
__global__ void __launch_bounds__(256) k_sweep_fold(const FoldSweepArgs a)
{
    const FoldGeom f = a.f;
    const int M = MT ? MT : f.M, K = MT ? 64 / MT : f.K;
    const unsigned L = a.lat.L, Lh = a.lat.Lh, W = Lh >> 1, Lz = f.Lz;
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= f.Nhf / 2) return;
    unsigned k, y, z; // z = folded plane
    if (POW2) {
        k = tid & (W - 1);
        const unsigned row = tid >> (a.lat.log2Lh - 1);
        y = row & (L - 1);
        z = row >> a.lat.log2L;
    } else {
        k = tid % W;
        const unsigned row = tid / W;
        y = row % L;
        z = row / L;
    }
    const unsigned s = (a.colour ^ (y + z)) & 1u;
    const unsigned yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const bool top = z + 1 == Lz, bottom = z == 0;
    const unsigned zp = top ? 0 : z + 1, zm = bottom ? Lz - 1 : z - 1;
    const unsigned rowbase = Lh * (y + L * z), i0 = rowbase + 2 * k;
    const unsigned xe = s ? ((2 * k + 2 == Lh) ? 0 : 2 * k + 2) : ((k == 0) ? Lh - 1 : 2 * k - 1);
    const unsigned ie = rowbase + xe;
    const unsigned iyp = Lh * (yp + L * z) + 2 * k, iym = Lh * (ym + L * z) + 2 * k;
    const unsigned izp = Lh * (y + L * zp) + 2 * k, izm = Lh * (y + L * zm) + 2 * k;
    const unsigned Nhf = f.Nhf;

    const ulonglong2 own = *(const ulonglong2 *)(a.own + i0);
    const ulonglong2 A = *(const ulonglong2 *)(a.oth + i0);
    const uint64_t ex = a.oth[ie];
    const ulonglong2 Yp = *(const ulonglong2 *)(a.oth + iyp), Ym = *(const ulonglong2 *)(a.oth + iym);
    ulonglong2 Zp = *(const ulonglong2 *)(a.oth + izp), Zm = *(const ulonglong2 *)(a.oth + izm);
    const ulonglong2 jx = *(const ulonglong2 *)(a.Jc + i0), jy = *(const ulonglong2 *)(a.Jc + Nhf + i0),
                     jz = *(const ulonglong2 *)(a.Jc + 2 * Nhf + i0);
    const ulonglong2 B = *(const ulonglong2 *)(a.Jo + i0);
    const uint64_t Jex = a.Jo[ie];
    const ulonglong2 by = *(const ulonglong2 *)(a.Jo + Nhf + iym);
    ulonglong2 bz = *(const ulonglong2 *)(a.Jo + 2 * Nhf + izm);
    if (top) { // slab k couples to slab k + 1 across the seam ("rotate the bits ... by M positions")
        Zp.x = rotr64(Zp.x, M); Zp.y = rotr64(Zp.y, M);
    }
    if (bottom) {
        Zm.x = rotl64(Zm.x, M); Zm.y = rotl64(Zm.y, M);
        bz.x = rotl64(bz.x, M); bz.y = rotl64(bz.y, M);
    }
    const uint64_t np0 = s ? A.y : A.x, nm0 = s ? A.x : ex;
    const uint64_t np1 = s ? ex : A.y, nm1 = s ? A.y : A.x;
    const uint64_t jm0 = s ? B.x : Jex, jm1 = s ? B.y : B.x;

    // level masks: K physical sites per word, each with its own numbers (keyed by the physical site; the thread's
    // two words are one pair of the stream contract C-A7)
    const uint64_t time = (a.d_time ? *a.d_time : a.t) + a.t_offset;
    const SweepRng g = make_sweep_rng(a.seed, time, (uint32_t)a.colour);
    uint64_t glo = f.g_lo, ghi = f.g_hi;                           // the slab's group bits, shifted by M per slab
    if (HB) {
        uint64_t ma[7], mb[7]; // word 0 (a), word 1 (b)
#pragma unroll
        for (int l = 0; l < 7; ++l) ma[l] = mb[l] = a.th.hb_always[l] ? ~(uint64_t)0 : 0; // hb[l] == 2^32 (T = 0): certain
        for (int kk = 0; kk < K; ++kk) {
            const uint32_t site0 = (4 * k + s) + L * (y + L * (z + kk * Lz));
            const uint4 r = sweep_random4(g, site0);
#pragma unroll
            for (int l = 0; l < 7; ++l) {
                if (r.x < a.th.hb[l]) ma[l] |= glo;
                if (r.y < a.th.hb[l]) ma[l] |= ghi;
                if (r.z < a.th.hb[l]) mb[l] |= glo;
                if (r.w < a.th.hb[l]) mb[l] |= ghi;
            }
            glo <<= M;
            ghi <<= M;
        }
        ulonglong2 out;
        out.x = own.x ^ flip_word_masks_heatbath(own.x, np0, nm0, Yp.x, Ym.x, Zp.x, Zm.x, jx.x, jm0, jy.x, by.x, jz.x, bz.x, ma);
        out.y = own.y ^ flip_word_masks_heatbath(own.y, np1, nm1, Yp.y, Ym.y, Zp.y, Zm.y, jx.y, jm1, jy.y, by.y, jz.y, bz.y, mb);
        *(ulonglong2 *)(a.own + i0) = out;
        return;
    }
    uint64_t m0a = 0, m1a = 0, m2a = 0, m0b = 0, m1b = 0, m2b = 0; // word 0 (a), word 1 (b)
#pragma unroll(MT ? (64 / (MT ? MT : 1) <= 8 ? 64 / (MT ? MT : 1) : 4) : 1)
    for (int kk = 0; kk < K; ++kk) {
        const uint32_t site0 = (4 * k + s) + L * (y + L * (z + kk * Lz));
        const uint4 r = sweep_random4(g, site0);
        // energy-raising moves are rare at low T: one branch per slab skips all the mask work when none of the four
        // numbers is below thr[2] (thr[0] <= thr[1] <= thr[2])
        if (ALWAYS || min(min(r.x, r.y), min(r.z, r.w)) < a.th.thr[2]) {
            if (r.x < a.th.thr[2]) m2a |= glo;
            if (r.y < a.th.thr[2]) m2a |= ghi;
            if (r.z < a.th.thr[2]) m2b |= glo;
            if (r.w < a.th.thr[2]) m2b |= ghi;
            if (r.x < a.th.thr[1]) m1a |= glo;
            if (r.y < a.th.thr[1]) m1a |= ghi;
            if (r.z < a.th.thr[1]) m1b |= glo;
            if (r.w < a.th.thr[1]) m1b |= ghi;
            if (r.x < a.th.thr[0]) m0a |= glo;
            if (r.y < a.th.thr[0]) m0a |= ghi;
            if (r.z < a.th.thr[0]) m0b |= glo;
            if (r.w < a.th.thr[0]) m0b |= ghi;
        }
        glo <<= M;
        ghi <<= M;
    }
    if (ALWAYS) { // thr[k] == 2^32 (T = inf): certain, whatever the number
        const uint64_t al0 = a.th.always[0] ? ~(uint64_t)0 : 0, al1 = a.th.always[1] ? ~(uint64_t)0 : 0, al2 = a.th.always[2] ? ~(uint64_t)0 : 0;
        m0a |= al0; m0b |= al0; m1a |= al1; m1b |= al1; m2a |= al2; m2b |= al2;
    }
    ulonglong2 out;
    out.x = own.x ^ flip_word_masks(own.x, np0, nm0, Yp.x, Ym.x, Zp.x, Zm.x, jx.x, jm0, jy.x, by.x, jz.x, bz.x, m0a, m1a, m2a);
    out.y = own.y ^ flip_word_masks(own.y, np1, nm1, Yp.y, Ym.y, Zp.y, Zm.y, jx.y, jm1, jy.y, by.y, jz.y, bz.y, m0b, m1b, m2b);
    *(ulonglong2 *)(a.own + i0) = out;
}

// ---------------------------------------------------------------------------------------------
static inline unsigned blocks_for(size_t n, unsigned block) { return (unsigned)((n + block - 1) / block); }

bool fold_valid(int L, int n_samples, int n_replicas)
{
    if (n_samples == 64) return true;
    if (n_samples < 1 || n_samples > 32 || (n_samples & (n_samples - 1))) return false;
    if (n_replicas == 2 && n_samples < 2) return false;
    const int K = 64 / n_samples;
    if (L % 4 || L % K) return false;
    const int Lz = L / K;
    return Lz >= 2 && Lz % 2 == 0;
}

size_t fold_bytes(int L, int n_samples)
{
    if (n_samples == 64) return 0;
    const size_t N = (size_t)L * L * L, K = 64 / n_samples;
    return (N / K + 3 * N / K) * 8; // folded spins + folded 64-bit bonds
}

// standard spins / bonds (complete, all 64 lanes as drawn) -> mask the unused lanes, build the folded copies
cudaError_t fold_from_standard(ea_sim *s, bool spins, bool bonds)
{
    const FoldGeom f = fold_geom(s);
    const unsigned Nh = s->lat.Nh;
    const uint64_t lane_mask = expand_lanes_host(s);
    if (spins) {
        k_mask_words<uint64_t><<<blocks_for(2 * (size_t)Nh, 256), 256, 0, s->stream>>>(s->spins, 2 * (size_t)Nh, lane_mask);
        k_fold_spins<<<blocks_for(2 * (size_t)f.Nhf, 256), 256, 0, s->stream>>>(f, Nh, s->spins, s->f_spins);
        s->count_launch(2);
        s->unfolded_valid = true;
    }
    if (bonds) {
        if (s->n_replicas == 2) {
            k_mask_words<uint32_t><<<blocks_for(6 * (size_t)Nh, 256), 256, 0, s->stream>>>((uint32_t *)s->bonds, 6 * (size_t)Nh, (uint32_t)lane_mask);
            k_fold_bonds<uint32_t><<<blocks_for(6 * (size_t)f.Nhf, 256), 256, 0, s->stream>>>(f, Nh, (const uint32_t *)s->bonds, s->f_bonds);
        } else {
            k_mask_words<uint64_t><<<blocks_for(6 * (size_t)Nh, 256), 256, 0, s->stream>>>((uint64_t *)s->bonds, 6 * (size_t)Nh, lane_mask);
            k_fold_bonds<uint64_t><<<blocks_for(6 * (size_t)f.Nhf, 256), 256, 0, s->stream>>>(f, Nh, (const uint64_t *)s->bonds, s->f_bonds);
        }
        s->count_launch(2);
    }
    return cudaGetLastError();
}

// the 64-lane mask of the samples a folded sim carries (C-M)
uint64_t expand_lanes_host(const ea_sim *s)
{
    if (s->n_samples == 64) return ~(uint64_t)0;
    const int M = s->n_samples;
    if (s->n_replicas == 2) {
        const uint64_t h = ((uint64_t)1 << (M / 2)) - 1;
        return h | (h << 32);
    }
    return ((uint64_t)1 << M) - 1;
}

// make the standard-layout spin array current (observables, snapshots and ea_get_spins read it)
cudaError_t fold_ensure_unfolded(ea_sim *s)
{
    if (s->n_samples == 64 || s->unfolded_valid) return cudaSuccess;
    const FoldGeom f = fold_geom(s);
    k_unfold_spins<<<blocks_for(2 * (size_t)f.Nhf, 256), 256, 0, s->stream>>>(f, s->lat.Nh, s->f_spins, s->spins);
    s->count_launch();
    s->unfolded_valid = true;
    return cudaGetLastError();
}

cudaError_t launch_half_sweep_fold(ea_sim *s, int parity, uint64_t t, const uint64_t *d_time, uint32_t t_offset, cudaStream_t st)
{
    FoldSweepArgs a;
    a.f = fold_geom(s);
    a.lat = s->lat;
    a.colour = parity;
    a.own = s->f_spins + (size_t)parity * a.f.Nhf;
    a.oth = s->f_spins + (size_t)(1 - parity) * a.f.Nhf;
    a.Jc = s->f_bonds + (size_t)parity * 3 * a.f.Nhf;
    a.Jo = s->f_bonds + (size_t)(1 - parity) * 3 * a.f.Nhf;
    a.seed = s->seed;
    a.t = t;
    a.d_time = d_time;
    a.t_offset = t_offset;
    a.th = s->th;
    const bool always = a.th.always[0] | a.th.always[1] | a.th.always[2];
    const unsigned grid = blocks_for(a.f.Nhf / 2, 256);
    if (s->dynamics == EA_DYN_HEATBATH) { // the generic kernel with seven level masks
        k_sweep_fold<0, false, false, true><<<grid, 256, 0, st>>>(a);
    } else if (always || s->lat.log2L < 0) { // T = inf or L not a power of two: the generic kernel
        if (always) k_sweep_fold<0, false, true><<<grid, 256, 0, st>>>(a);
        else k_sweep_fold<0, false, false><<<grid, 256, 0, st>>>(a);
    } else {
        switch (a.f.M) {
        case 32: k_sweep_fold<32, true, false><<<grid, 256, 0, st>>>(a); break;
        case 16: k_sweep_fold<16, true, false><<<grid, 256, 0, st>>>(a); break;
        case 8: k_sweep_fold<8, true, false><<<grid, 256, 0, st>>>(a); break;
        case 4: k_sweep_fold<4, true, false><<<grid, 256, 0, st>>>(a); break;
        default: k_sweep_fold<0, true, false><<<grid, 256, 0, st>>>(a); break;
        }
    }
    s->count_launch();
    s->unfolded_valid = false;
    return cudaGetLastError();
}

} // namespace ea

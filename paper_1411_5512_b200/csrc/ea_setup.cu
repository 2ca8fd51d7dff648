// ea_setup.cu -- lattice setup (random bonds, random start) and the canonical <-> internal layout kernels.
#include "ea_internal.h"

namespace ea {

// canonical site of (colour c, compact index i)
__device__ __forceinline__ uint32_t canonical_site(const Lattice &lat, unsigned c, unsigned i)
{
    unsigned xh = i % lat.Lh, row = i / lat.Lh; // row = y + L*z
    unsigned y = row % lat.L, z = row / lat.L;
    unsigned x = 2 * xh + ((c ^ (y + z)) & 1u);
    return x + lat.L * row;
}

// (colour, compact index) of canonical site
__device__ __forceinline__ void compact_of(const Lattice &lat, unsigned site, unsigned &c, unsigned &i)
{
    unsigned x = site % lat.L, row = site / lat.L;
    unsigned y = row % lat.L, z = row / lat.L;
    c = (x + y + z) & 1u;
    i = (x >> 1) + lat.Lh * row;
}

// Random start = quench from T = inf.  C-A8: word(site) = out[0] | out[1] << 32 of
// Philox(counter (site, 0, 0, 2); key = seed).
__global__ void k_init_spins(Lattice lat, uint64_t *spins, uint64_t seed)
{
    unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= 2 * lat.Nh) return;
    unsigned c = tid >= lat.Nh, i = tid - c * lat.Nh;
    uint32_t out[4];
    philox4x32_10(canonical_site(lat, c, i), 0u, 0u, TAG_INIT_SPINS, (uint32_t)seed, (uint32_t)(seed >> 32), out);
    spins[tid] = mk64(out[0], out[1]);
}

// Bonds iid from P(J) = p delta(J-1) + (1-p) delta(J+1).  C-A9: P = floor(2^32 p + 0.5);
// sample b of bond (d, site): v = out[b & 3] of Philox(counter (site, 16 d + (b >> 2), 0, 3)); J = +1 (bit 0)
// iff v < P.  BondT = uint32: 32 disorder samples, shared by the two replicas.
template <typename BondT>
__global__ void k_init_bonds(Lattice lat, BondT *bonds, uint64_t seed, uint64_t P)
{
    unsigned tid = blockIdx.x * blockDim.x + threadIdx.x; // over [2][3][Nh]
    if (tid >= 6 * lat.Nh) return;
    unsigned c = tid / (3 * lat.Nh), rem = tid - c * 3 * lat.Nh;
    unsigned d = rem / lat.Nh, i = rem - d * lat.Nh;
    uint32_t site = canonical_site(lat, c, i);
    BondT w = 0;
    constexpr int BLOCKS = sizeof(BondT) * 2; // 4 samples per Philox block
    for (int q = 0; q < BLOCKS; ++q) {
        uint32_t out[4];
        philox4x32_10(site, 16u * d + q, 0u, TAG_BONDS, (uint32_t)seed, (uint32_t)(seed >> 32), out);
#pragma unroll
        for (int e = 0; e < 4; ++e)
            if (!((uint64_t)out[e] < P)) w |= (BondT)1 << (4 * q + e); // bit 1 <-> J = -1 (C-A2)
    }
    bonds[tid] = w;
}

__global__ void k_pack_spins(Lattice lat, const uint64_t *canon, uint64_t *internal)
{
    unsigned site = blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= 2 * lat.Nh) return;
    unsigned c, i;
    compact_of(lat, site, c, i);
    internal[(size_t)c * lat.Nh + i] = canon[site];
}

__global__ void k_unpack_spins(Lattice lat, const uint64_t *internal, uint64_t *canon)
{
    unsigned site = blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= 2 * lat.Nh) return;
    unsigned c, i;
    compact_of(lat, site, c, i);
    canon[site] = internal[(size_t)c * lat.Nh + i];
}

// bad != nullptr (32-bit bond words): raise *bad if a word's hi half differs from its lo half -- both replicas must
// have "the same bond configuration"; checked here instead of in a host loop over 3 N words
template <typename BondT>
__global__ void k_pack_bonds(Lattice lat, unsigned d, const uint64_t *canon, BondT *bonds, unsigned *bad)
{
    unsigned site = blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= 2 * lat.Nh) return;
    unsigned c, i;
    compact_of(lat, site, c, i);
    const uint64_t w = canon[site];
    if (sizeof(BondT) == 4 && bad && lo32(w) != hi32(w)) atomicOr(bad, 1u);
    bonds[((size_t)c * 3 + d) * lat.Nh + i] = (BondT)w;
}

template <typename BondT>
__global__ void k_unpack_bonds(Lattice lat, unsigned d, const BondT *bonds, uint64_t *canon)
{
    unsigned site = blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= 2 * lat.Nh) return;
    unsigned c, i;
    compact_of(lat, site, c, i);
    BondT w = bonds[((size_t)c * 3 + d) * lat.Nh + i];
    canon[site] = sizeof(BondT) == 4 ? mk64((uint32_t)w, (uint32_t)w) : (uint64_t)w;
}

__global__ void k_philox_selftest(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                  uint32_t *out)
{
    uint32_t o[4];
    philox4x32_10(c0, c1, c2, c3, k0, k1, o);
    for (int e = 0; e < 4; ++e) out[e] = o[e];
    // the folded update stream must agree with the block function: out[4..7] = sweep_random4 of the same counter
    SweepRng g = make_sweep_rng((uint64_t)k0 | ((uint64_t)k1 << 32), (uint64_t)c1 | ((uint64_t)c2 << 32), c3);
    const uint4 f = sweep_random4(g, c0);
    out[4] = f.x; out[5] = f.y; out[6] = f.z; out[7] = f.w;
}

static inline unsigned blocks_for(size_t n, unsigned block) { return (unsigned)((n + block - 1) / block); }

cudaError_t launch_init_spins(ea_sim *s)
{
    size_t n = 2 * (size_t)s->lat.Nh;
    k_init_spins<<<blocks_for(n, 256), 256, 0, s->stream>>>(s->lat, s->spins, s->seed);
    s->count_launch();
    return cudaGetLastError();
}

// floor(2^32 p + 0.5) as an integer in [0, 2^32] (C-A9)
static uint64_t bond_threshold(double p) { return (uint64_t)(4294967296.0 * p + 0.5); }

cudaError_t launch_init_bonds(ea_sim *s)
{
    size_t n = 6 * (size_t)s->lat.Nh;
    uint64_t P = bond_threshold(s->p);
    if (s->n_replicas == 2)
        k_init_bonds<uint32_t><<<blocks_for(n, 256), 256, 0, s->stream>>>(s->lat, (uint32_t *)s->bonds, s->seed, P);
    else
        k_init_bonds<uint64_t><<<blocks_for(n, 256), 256, 0, s->stream>>>(s->lat, (uint64_t *)s->bonds, s->seed, P);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pack_spins(ea_sim *s, const uint64_t *d_canon, uint64_t *d_internal)
{
    k_pack_spins<<<blocks_for(s->N, 256), 256, 0, s->stream>>>(s->lat, d_canon, d_internal);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_unpack_spins(ea_sim *s, const uint64_t *d_internal, uint64_t *d_canon)
{
    k_unpack_spins<<<blocks_for(s->N, 256), 256, 0, s->stream>>>(s->lat, d_internal, d_canon);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pack_bonds(ea_sim *s, int d, const uint64_t *d_canon, unsigned *d_bad)
{
    if (s->n_replicas == 2)
        k_pack_bonds<uint32_t><<<blocks_for(s->N, 256), 256, 0, s->stream>>>(s->lat, d, d_canon, (uint32_t *)s->bonds, d_bad);
    else
        k_pack_bonds<uint64_t><<<blocks_for(s->N, 256), 256, 0, s->stream>>>(s->lat, d, d_canon, (uint64_t *)s->bonds, nullptr);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t launch_unpack_bonds(ea_sim *s, int d, uint64_t *d_canon)
{
    if (s->n_replicas == 2)
        k_unpack_bonds<uint32_t><<<blocks_for(s->N, 256), 256, 0, s->stream>>>(s->lat, d, (const uint32_t *)s->bonds, d_canon);
    else
        k_unpack_bonds<uint64_t><<<blocks_for(s->N, 256), 256, 0, s->stream>>>(s->lat, d, (const uint64_t *)s->bonds, d_canon);
    s->count_launch();
    return cudaGetLastError();
}

cudaError_t philox_selftest(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t *d = nullptr, h[8];
    cudaError_t e = cudaMalloc(&d, sizeof(h));
    if (e != cudaSuccess) return e;
    k_philox_selftest<<<1, 1>>>(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1], d);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return e;
    // the folded stream is only defined for tags 0/1 but the algebra holds for any counter: require agreement
    if (h[4] != h[0] || h[5] != h[1] || h[6] != h[2] || h[7] != h[3]) return cudaErrorUnknown;
    for (int i = 0; i < 4; ++i) out[i] = h[i];
    return cudaSuccess;
}

} // namespace ea

// ea_sweep_small.cu -- SMALL: the whole lattice in shared memory for the n sweeps of one ea_sweep(n) call, for the
// small lattices of the paper's scans (L = 8 .. 32: PAPER.md:134 and BASELINE configs 1-2), where a kernel launch
// per colour costs far more than the half-sweep itself.
//
// Same update and the same stream contract as every other variant, hence bit-identical.  The lattice is cut into
// C = Cy x Cz blocks of L x (L / Cy) x (L / Cz) sites (whole x rows), one CTA per block:
//   * C = 1 (L <= 8): one CTA, the colour barrier is __syncthreads();
//   * C = 2 .. 16 (L = 32: 16 slabs of 2 planes; L = 20, 24: 4 x 4 blocks): one thread-block CLUSTER; a thread on a face of
//     its block PUSHES its new pair into the halo of the neighbouring CTA's shared memory (st.async through distributed
//     shared memory) and the colour barrier is an mbarrier per CTA that counts its own warps and the bytes its neighbours
//     pushed -- no global memory traffic, no cluster-wide barrier and no fence wider than the CTA between sweeps (PUSH below).
// Spins AND bond words live in shared memory; global memory is read once at the start and written once at the end.
// A thread owns one pair of x-adjacent same-colour sites of each colour (one Philox block per pair and sweep, C-A7).
#include <stdlib.h>

#include "ea_internal.h"
#include "ea_sweep_common.cuh"

namespace ea {

struct SmallArgs {
    uint64_t *spins;     // [2][Nh]
    const void *bonds;   // BondT [2][3][Nh]
    uint64_t seed;
    uint64_t t0;         // first sweep index
    uint32_t n_half;     // half-sweeps to run
    int L, Ly, Lz;       // side; rows and planes per CTA
    int Cy, Cz;          // CTAs along y and z (Cy Cz = cluster size; rank = ry + Cy rz)
    Thresholds th;
};

__device__ __forceinline__ uint32_t small_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// address of the same shared-memory location in the CTA of rank `rank` of this cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared-memory loads by 32-bit shared address (precomputed once per thread: the sweep loop holds no index arithmetic)
__device__ __forceinline__ uint64_t lds_u64(uint32_t addr)
{
    uint64_t v;
    asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ ulonglong2 lds_v2u64(uint32_t addr)
{
    ulonglong2 v;
    asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr) : "memory");
    return v;
}
// the thread's twelve bond words of one colour: BondT [12 sizeof(BondT) / 16][n_threads] vectors of 16 bytes, so that every
// load is one conflict-free LDS.128 of the warp
__device__ __forceinline__ void lds_bonds12(uint32_t addr, uint32_t stride, uint32_t (&j)[12])
{
#pragma unroll
    for (int k = 0; k < 3; ++k)
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(j[4 * k]), "=r"(j[4 * k + 1]), "=r"(j[4 * k + 2]), "=r"(j[4 * k + 3])
                     : "r"(addr + k * stride) : "memory");
}
__device__ __forceinline__ void lds_bonds12(uint32_t addr, uint32_t stride, uint64_t (&j)[12])
{
#pragma unroll
    for (int k = 0; k < 6; ++k)
        asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(j[2 * k]), "=l"(j[2 * k + 1]) : "r"(addr + k * stride) : "memory");
}
__device__ __forceinline__ void sts_v2u64(uint32_t addr, ulonglong2 v)
{
    asm volatile("st.shared.v2.u64 [%0], {%1, %2};" ::"r"(addr), "l"(v.x), "l"(v.y) : "memory");
}

// mbarrier of the push exchange (PUSH): local arrivals of the CTA's warps + the bytes the two neighbours push
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "WAIT_%=:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@!p bra WAIT_%=;\n"
                 "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// 16 bytes into a neighbouring CTA's shared memory; the bytes are counted on that CTA's mbarrier when they have landed
__device__ __forceinline__ void st_async_v2u64(uint32_t remote, ulonglong2 v, uint32_t remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];" ::"r"(remote), "l"(v.x),
                 "l"(v.y), "r"(remote_bar) : "memory");
}

// Shared-memory addresses of everything one half-sweep of colour c touches for the thread's pair
struct SmallAddr {
    uint32_t own, xa, xe, pm, pp, zm, zp;       // spins: own pair; the other colour's pair at the same place and the row's third
                                                // other-colour word next to it; y -/+ and z -/+ pairs
    uint32_t bonds;                             // the thread's bond vectors of this colour
    uint32_t push_zlo, push_zhi, push_ylo, push_yhi; // PUSH: where the own pair goes in the CTA below / above along z and y
                                                // (shared::cluster addresses)
};

__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// (only at the start and the end of the kernel: see PUSH)

// Shared memory of one CTA (Ly x Lz rows of Lh = L / 2 words per colour; nh = Lh Ly Lz words per colour of the block):
//   spins  uint64 [2][Lz][Ly][Lh]
//   bonds  BondT  [2][12][n_threads] in vectors of 16 bytes: per colour and thread {jx, jx', jy, jy', jz, jz', bl, bl', by, by',
//                 bz, bz'} = the forward bonds of the pair's two sites, the +x bonds of their left neighbours, the +y / +z bonds of
//                 their y - 1 / z - 1 neighbours.  Every bond sits there twice (forward for one colour, backward for the other):
//                 the addresses never change, so each thread keeps its own copy where one LDS.128 per four words fetches it.
//   zhalo  uint64 [2][2][Ly][Lh]  PUSH: the faces below / above the block along z, both colours, as the neighbours pushed them
//   yhalo  uint64 [2][2][Lz][Lh]  PUSH, Cy > 1 (YSPLIT): the same along y
//   bar    uint64 [2]             PUSH: one mbarrier per colour
//
// PUSH (clusters): no cluster barrier in the sweep loop.  barrier.cluster.arrive.release / wait.acquire compile to
// MEMBAR.ALL.GPU + UCGABAR + CCTL.IVALL (measured ~850 clocks per barrier on 8 CTAs, ~1240 on 16), and so does every other
// release / acquire at cluster scope (remote mbarrier arrives were slower still).  Instead a thread on a boundary plane
// stores its new pair into its own slab AND into the facing halo plane of the neighbouring CTA with st.async (STAS), which
// counts the bytes on that CTA's mbarrier when they have landed; the warps of a CTA arrive on the same mbarrier after
// their stores.  A half-sweep of colour c completes phase (sweep & 1) of bar[c]; everybody waits on it before the next
// half-sweep and reads only LOCAL shared memory.  Hazards: a halo word is rewritten two half-sweeps later, which the
// neighbour starts only after THIS CTA's pushes of the half-sweep between, each made by the thread that read the word.
// Measured (B200, us per half-sweep, L = 16 / 32): cluster barrier + remote loads 0.59 / 1.03; pushes 0.36 / 0.71.  Not
// kept: cp.async.bulk of the whole plane by one thread (0.50 / 1.00: the copy starts only after a CTA-wide barrier), two
// interleaved chains of row classes as in the L = 128 kernel (0.69 at L = 32: a unit's latency, not its issue slots, sets
// the pace).  The number of pushed pairs does not matter either (see small_shape).
template <typename BondT, bool ALWAYS, bool RARE, bool HB, bool CLUSTER, bool YSPLIT>
__global__ void __launch_bounds__(CLUSTER ? 512 : 128, 1) k_sweep_small(const SmallArgs a)
{
    constexpr bool PUSH = CLUSTER;
    extern __shared__ __align__(16) unsigned char smem_small[];
    const unsigned L = a.L, Lh = L / 2, Ly = a.Ly, Lz = a.Lz, hp = Lh / 2; // hp: pairs per row
    const unsigned Cy = a.Cy, Cz = a.Cz;
    const unsigned pz = Ly * Lh, py = Lz * Lh;  // words per colour of one z face (a plane of the block) / one y face
    const unsigned nh = pz * Lz, Nh = L * L * Lh;
    const unsigned rank = CLUSTER ? cluster_ctarank() : 0;
    const unsigned ry = rank % Cy, rz = rank / Cy, y0 = ry * Ly, z0 = rz * Lz;
    const bool split_y = YSPLIT, split_z = PUSH && (!YSPLIT || Cz > 1); // YSPLIT: Cy > 1 (compiled out of the slab variant)
    uint64_t *spins_s = (uint64_t *)smem_small;                // [2][Lz][Ly][Lh]
    const unsigned tid = threadIdx.x, nthr = blockDim.x;
    BondT *bonds_s = (BondT *)(spins_s + 2 * nh);
    uint64_t *zhalo_s = (uint64_t *)(bonds_s + 24 * nthr);     // [2 sides][2 colours][Ly][Lh]
    uint64_t *yhalo_s = zhalo_s + 4 * pz;                      // [2 sides][2 colours][Lz][Lh]
    uint64_t *bar_s = yhalo_s + 4 * py;
    const BondT *__restrict__ gb = (const BondT *)a.bonds;

    // ---- prologue: the block (whole x rows) and the four faces around it ------------------------------------------
    for (unsigned v = tid; v < 2 * nh; v += nthr) {
        const unsigned c = v / nh, i = v % nh, x = i % Lh, yl = (i / Lh) % Ly, zl = i / pz;
        spins_s[v] = a.spins[(size_t)c * Nh + (size_t)Lh * ((y0 + yl) + (size_t)L * (z0 + zl)) + x];
    }
    if (PUSH) {
        for (unsigned v = tid; v < 4 * pz; v += nthr) {
            const unsigned side = v / (2 * pz), c = (v / pz) & 1u, i = v % pz, x = i % Lh, yl = i / Lh;
            const unsigned zh = side ? (z0 + Lz) % L : (z0 + L - 1) % L;
            zhalo_s[v] = a.spins[(size_t)c * Nh + (size_t)Lh * ((y0 + yl) + (size_t)L * zh) + x];
        }
        for (unsigned v = tid; v < 4 * py; v += nthr) {
            const unsigned side = v / (2 * py), c = (v / py) & 1u, i = v % py, x = i % Lh, zl = i / Lh;
            const unsigned yh = side ? (y0 + Ly) % L : (y0 + L - 1) % L;
            yhalo_s[v] = a.spins[(size_t)c * Nh + (size_t)Lh * (yh + (size_t)L * (z0 + zl)) + x];
        }
        if (tid == 0) {
            mbar_init(small_smem_u32(bar_s), nthr / 32);
            mbar_init(small_smem_u32(bar_s + 1), nthr / 32);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }

    // ---- the thread's pair: (p, yl, zl) -> compact words 2p, 2p + 1 of row (yl, zl) of the block, both colours -----
    const unsigned n_pairs = hp * Ly * Lz;
    const bool active = tid < n_pairs;
    const unsigned p = tid % hp, yl = (tid / hp) % Ly, zl = active ? tid / (hp * Ly) : 0;
    const unsigned y = y0 + yl, zg = z0 + zl;                       // global row
    const unsigned ym = y == 0 ? L - 1 : y - 1;
    const unsigned rowb = Lh * (yl + Ly * zl), i0 = rowb + 2 * p;   // own words (and the other colour's words of the same position)
    // y / z neighbours: inside the block, or the facing halo (the neighbouring CTA's face); an unsplit direction wraps
    const bool ylo = yl == 0, yhi = yl + 1 == Ly, zlo = zl == 0, zhi = zl + 1 == Lz;
    const unsigned i_ym = Lh * ((ylo ? Ly - 1 : yl - 1) + Ly * zl) + 2 * p, i_yp = Lh * ((yhi ? 0 : yl + 1) + Ly * zl) + 2 * p;
    const unsigned i_zm = Lh * (yl + Ly * (zlo ? Lz - 1 : zl - 1)) + 2 * p, i_zp = Lh * (yl + Ly * (zhi ? 0 : zl + 1)) + 2 * p;
    const unsigned i_zf = Lh * yl + 2 * p, i_yf = Lh * zl + 2 * p;  // the pair inside a z face / a y face
    const uint32_t spins_a = small_smem_u32(spins_s);
    const uint32_t zhalo_a = small_smem_u32(zhalo_s), yhalo_a = small_smem_u32(yhalo_s), bar_a = small_smem_u32(bar_s);
    // the four neighbouring CTAs of the cluster (rank = ry + Cy rz)
    const unsigned r_zlo = ry + Cy * ((rz + Cz - 1) % Cz), r_zhi = ry + Cy * ((rz + 1) % Cz);
    const unsigned r_ylo = (ry + Cy - 1) % Cy + Cy * rz, r_yhi = (ry + 1) % Cy + Cy * rz;
    const uint32_t zhalo_zlo = PUSH ? mapa_u32(zhalo_a, r_zlo) : 0, zhalo_zhi = PUSH ? mapa_u32(zhalo_a, r_zhi) : 0;
    const uint32_t yhalo_ylo = PUSH ? mapa_u32(yhalo_a, r_ylo) : 0, yhalo_yhi = PUSH ? mapa_u32(yhalo_a, r_yhi) : 0;
    const uint32_t bar_zlo = PUSH ? mapa_u32(bar_a, r_zlo) : 0, bar_zhi = PUSH ? mapa_u32(bar_a, r_zhi) : 0;
    const uint32_t bar_ylo = PUSH ? mapa_u32(bar_a, r_ylo) : 0, bar_yhi = PUSH ? mapa_u32(bar_a, r_yhi) : 0;
    const bool push_zlo = split_z && zlo, push_zhi = split_z && zhi, push_ylo = split_y && ylo, push_yhi = split_y && yhi;
    const uint32_t site_row = L * (y + L * zg);

    // per colour c: x-phase S = (c ^ y ^ z) & 1; the three other-colour words of the row next to the pair are compact
    // q, q + 1, q + 2 with q = 2p - 1 + S (periodic)
    unsigned Sc[2];
    SmallAddr A[2];
    const uint32_t bonds_a = small_smem_u32(bonds_s);
    constexpr unsigned BS = sizeof(BondT), VEC = 16 / BS; // bond words per 16-byte vector
    const uint32_t bond_stride = 16 * nthr;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        Sc[c] = (c ^ y ^ zg) & 1u;
        const unsigned q0 = (2 * p + Sc[c] + Lh - 1) % Lh, q1 = (q0 + 1) % Lh, q2 = (q1 + 1) % Lh;
        const unsigned own_w = c * nh, oth_w = (1 - c) * nh;
        A[c].own = spins_a + (own_w + i0) * 8;
        A[c].xa = spins_a + (oth_w + i0) * 8;
        A[c].xe = spins_a + (oth_w + rowb + (Sc[c] ? q2 : q0)) * 8;
        A[c].pm = push_ylo ? yhalo_a + ((1 - c) * py + i_yf) * 8 : spins_a + (oth_w + i_ym) * 8;
        A[c].pp = push_yhi ? yhalo_a + ((2 + 1 - c) * py + i_yf) * 8 : spins_a + (oth_w + i_yp) * 8;
        A[c].zm = push_zlo ? zhalo_a + ((1 - c) * pz + i_zf) * 8 : spins_a + (oth_w + i_zm) * 8;
        A[c].zp = push_zhi ? zhalo_a + ((2 + 1 - c) * pz + i_zf) * 8 : spins_a + (oth_w + i_zp) * 8;
        A[c].push_zlo = zhalo_zlo + ((2 + c) * pz + i_zf) * 8; // the block's first plane is the face ABOVE the CTA below
        A[c].push_zhi = zhalo_zhi + (c * pz + i_zf) * 8;
        A[c].push_ylo = yhalo_ylo + ((2 + c) * py + i_yf) * 8;
        A[c].push_yhi = yhalo_yhi + (c * py + i_yf) * 8;
        A[c].bonds = bonds_a + c * (12 / VEC) * bond_stride + 16 * tid;
        if (active) { // the thread's copy of its bonds, straight from the global arrays [2][3][Nh]
            const size_t g_row = (size_t)Lh * (y + (size_t)L * zg), g_ym = (size_t)Lh * (ym + (size_t)L * zg);
            const size_t g_zm = (size_t)Lh * (y + (size_t)L * ((zg + L - 1) % L));
            const BondT *jc = gb + (size_t)c * 3 * Nh, *jo = gb + (size_t)(1 - c) * 3 * Nh;
            // +x bonds: jx / jx' of the own sites (towards compact q1 / q2), bl / bl' of their left neighbours q0 / q1
            const BondT jx = jc[g_row + 2 * p], jx2 = jc[g_row + 2 * p + 1], bl = jo[g_row + q0], bl2 = jo[g_row + q1];
            const bool S = Sc[c];
            const BondT w[12] = {S ? bl : jx, S ? bl2 : jx2, jc[Nh + g_row + 2 * p], jc[Nh + g_row + 2 * p + 1],
                                 jc[2 * (size_t)Nh + g_row + 2 * p], jc[2 * (size_t)Nh + g_row + 2 * p + 1],
                                 S ? jx : bl, S ? jx2 : bl2,
                                 jo[Nh + g_ym + 2 * p], jo[Nh + g_ym + 2 * p + 1],
                                 jo[2 * (size_t)Nh + g_zm + 2 * p], jo[2 * (size_t)Nh + g_zm + 2 * p + 1]};
#pragma unroll
            for (int k = 0; k < 12; ++k) bonds_s[((size_t)c * (12 / VEC) + k / VEC) * VEC * nthr + (size_t)VEC * tid + k % VEC] = w[k];
        }
    }
    const uint32_t site0 = site_row + 4 * p + Sc[0], site1 = site_row + 4 * p + Sc[1]; // first site of the pair, colour 0 / 1

    // the thread's own pairs stay in registers between the sweeps (nobody else writes them); shared memory holds the copy
    // the neighbours read
    ulonglong2 own_r[2] = {};
    auto half_sweep = [&](const SmallAddr &ad, const uint4 r, const unsigned c, const bool S, const BondT (&j)[12]) {
        // the row's other-colour words next to the pair: compact q0, q0 + 1, q0 + 2 with q0 = 2p - 1 + S
        const ulonglong2 Xa = lds_v2u64(ad.xa);
        const uint64_t Xe = lds_u64(ad.xe);
        // first word: x neighbours Xa.x and (S ? Xa.y : Xe); second word: Xa.y and (S ? Xe : Xa.x).  The thread's x-bond
        // words are stored in that order (the six terms of the local field are symmetric: only the pairing matters).
        const uint64_t A2 = S ? Xa.y : Xe, B2 = S ? Xe : Xa.x;
        const ulonglong2 own = own_r[c], Pm = lds_v2u64(ad.pm), Pp = lds_v2u64(ad.pp);
        const ulonglong2 Zm = lds_v2u64(ad.zm), Zp = lds_v2u64(ad.zp);
        const BondT xA1 = j[0], xB1 = j[1], jyA = j[2], jyB = j[3], jzA = j[4], jzB = j[5], xA2 = j[6], xB2 = j[7], byA = j[8],
                    byB = j[9], bzA = j[10], bzB = j[11];
        ulonglong2 out;
        out.x = metropolis_word<BondT, ALWAYS, RARE, HB>(own.x, Xa.x, A2, Pp.x, Pm.x, Zp.x, Zm.x, xA1, xA2, jyA, byA, jzA, bzA, r.x, r.y, a.th);
        out.y = metropolis_word<BondT, ALWAYS, RARE, HB>(own.y, Xa.y, B2, Pp.y, Pm.y, Zp.y, Zm.y, xB1, xB2, jyB, byB, jzB, bzB, r.z, r.w, a.th);
        if (active) sts_v2u64(ad.own, out);
        own_r[c] = out;
        if (PUSH) {
            if (push_zlo) st_async_v2u64(ad.push_zlo, out, bar_zlo + 8 * c);
            if (push_zhi) st_async_v2u64(ad.push_zhi, out, bar_zhi + 8 * c);
            if (push_ylo) st_async_v2u64(ad.push_ylo, out, bar_ylo + 8 * c);
            if (push_yhi) st_async_v2u64(ad.push_yhi, out, bar_yhi + 8 * c);
        }
    };

    // end of a half-sweep: arrive at the colour barrier, draw the next random numbers meanwhile, wait
    const uint32_t tx_bytes = (split_z ? 2 * pz * 8 : 0) + (split_y ? 2 * py * 8 : 0); // what the neighbours push per half-sweep
    auto barrier_begin = [&](const unsigned c) {
        if (PUSH) {
            __syncwarp();
            if (tid == 0) mbar_arrive_expect_tx(bar_a + 8 * c, tx_bytes);
            else if ((tid & 31u) == 0) mbar_arrive(bar_a + 8 * c);
        }
    };
    auto barrier_end = [&](const unsigned c, const uint32_t parity) {
        if (PUSH) mbar_wait(bar_a + 8 * c, parity);
        else __syncthreads();
    };

    SweepRng g = make_sweep_rng(a.seed, a.t0, 0);
    // the random numbers do not depend on the spins: those of the next half-sweep are drawn while the barrier completes
    uint4 r = sweep_random4(g, site0);
    if (CLUSTER) cluster_barrier(); else __syncthreads(); // every CTA of the cluster has its slab in place

    if (active) {
        own_r[0] = lds_v2u64(A[0].own);
        own_r[1] = lds_v2u64(A[1].own);
    }
    // The bond words do not depend on the exchange: those of the next half-sweep are fetched while the barrier completes, so
    // that only the spin loads queue on the load pipe when all warps start the half-sweep together (a trace showed ~600 clocks
    // from the first load to the last operand at L = 32, against ~500 of logic).
    BondT j[12];
    lds_bonds12(A[0].bonds, bond_stride, j);
    auto draw = [&](const uint64_t t, const uint32_t colour) {
        sweep_rng_set_time(g, t, colour);
        return sweep_random4(g, colour ? site1 : site0);
    };
    if (!CLUSTER && !HB) {
        // one CTA, one warp per sub-partition: nothing to overlap with but the warp's own instructions.  The next numbers
        // are drawn in the same basic block as the loads and the logic of the current half-sweep (no branch around the
        // update: only the store is predicated), so that the Philox chain fills the load and dependency latencies
        // (L = 8: 0.30 -> 0.25 us per half-sweep with 64-bit bond words, 0.28 -> 0.24 with 32-bit ones; the heat bath's seven
        // predicated levels did not gain).  Up to 255 registers: the one-CTA kernel never has more than 128 threads.
        BondT j1[12];
#pragma unroll 1
        for (uint32_t sw = 0; sw < a.n_half / 2; ++sw) {
            const uint4 r1 = draw(a.t0 + sw, 1u);
            lds_bonds12(A[1].bonds, bond_stride, j1);
            half_sweep(A[0], r, 0, Sc[0], j);
            __syncthreads();
            r = draw(a.t0 + sw + 1, 0u);
            lds_bonds12(A[0].bonds, bond_stride, j);
            half_sweep(A[1], r1, 1, Sc[1], j1);
            __syncthreads();
        }
    } else
    for (uint32_t sw = 0; sw < a.n_half / 2; ++sw) { // n_half is even: colour 0 then colour 1 of sweep t0 + sw
        if (active) half_sweep(A[0], r, 0, Sc[0], j);
        barrier_begin(0);
        r = draw(a.t0 + sw, 1u);
        lds_bonds12(A[1].bonds, bond_stride, j);
        barrier_end(0, sw & 1u);
        if (active) half_sweep(A[1], r, 1, Sc[1], j);
        barrier_begin(1);
        r = draw(a.t0 + sw + 1, 0u);
        lds_bonds12(A[0].bonds, bond_stride, j);
        barrier_end(1, sw & 1u);
    }
    if (CLUSTER) cluster_barrier(); // nobody leaves while a neighbour may still read its shared memory

    // ---- epilogue: the block back to global ---------------------------------------------------------------------------
    for (unsigned v = tid; v < 2 * nh; v += nthr) {
        const unsigned c = v / nh, i = v % nh, x = i % Lh, yl_ = (i / Lh) % Ly, zl_ = i / pz;
        a.spins[(size_t)c * Nh + (size_t)Lh * ((y0 + yl_) + (size_t)L * (z0 + zl_)) + x] = spins_s[v];
    }
}

// ---------------------------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------------------------
struct SmallShape {
    int Cy, Cz;   // CTAs along y and z; 0: no valid shape
    int C() const { return Cy * Cz; }
};

static size_t small_smem_bytes(int L, int Ly, int Lz, int bond_bytes)
{
    const size_t Lh = L / 2, nh = Lh * Ly * Lz, pz = Ly * Lh, py = Lz * Lh;
    const size_t threads = ((size_t)(L / 4) * Ly * Lz + 31) / 32 * 32;
    return 2 * nh * 8 + 24 * threads * bond_bytes + 4 * pz * 8 + 4 * py * 8 + 16; // spins, bonds, z and y halos, bar
}

// The cluster (Cy x Cz CTAs, 1 .. 16, blocks of L x L/Cy x L/Cz sites) for a lattice of side L: every block must fit one
// CTA (at most 512 pairs = threads, and the shared memory of one SM); among those the one with the smallest estimated
// half-sweep time -- warps per sub-partition x ~300 clocks per pair, plus ~40 clocks for __syncthreads() or ~450 for the
// exchange between CTAs (measured: whatever the number of pushed pairs -- L = 32 as 1 x 16, 2 x 8, 4 x 4 blocks: 0.72 / 0.75 /
// 0.76 us; the y split costs a little for its extra predicated pushes).  What the y split buys is sixteen CTAs for sides
// that are no power of two (L = 20: 0.59 -> 0.38 us, L = 24: 0.66 -> 0.52).  Cy = 0 if there is none.
static SmallShape small_shape(int L, int n_replicas)
{
    SmallShape best = {0, 0};
    if (L < 4 || L % 4 || L > 64) return best;
    // EA_SMALL_CY / EA_SMALL_CZ (both set): the shape, for measurements like the ones quoted above; shapes that do not fit are skipped
    static const int forced_cy = [] { const char *e = getenv("EA_SMALL_CY"); return e ? atoi(e) : 0; }();
    static const int forced_cz = [] { const char *e = getenv("EA_SMALL_CZ"); return e ? atoi(e) : 0; }();
    const int bond_bytes = n_replicas == 2 ? 4 : 8, hp = L / 4;
    long best_cost = 0;
    for (int C = 1; C <= 16; C *= 2)
        for (int Cy = 1; Cy <= C; Cy *= 2) {
            const int Cz = C / Cy;
            if (L % Cy || L % Cz) continue;
            if (forced_cy && forced_cz && (Cy != forced_cy || Cz != forced_cz)) continue;
            const int Ly = L / Cy, Lz = L / Cz;
            const long pairs = (long)hp * Ly * Lz;
            if (pairs > (C == 1 ? 128 : 512) || small_smem_bytes(L, Ly, Lz, bond_bytes) > 200 * 1024) continue; // launch bounds
            const long cost = (pairs + 127) / 128 * 300 + (Cy * Cz == 1 ? 40 : Cy == 1 ? 450 : 510);
            if (!best.Cy || cost < best_cost) { best.Cy = Cy; best.Cz = Cz; best_cost = cost; } // ties: the smaller cluster
        }
    return best;
}

int small_cluster_size(int L, int n_replicas)
{
    const SmallShape sh = small_shape(L, n_replicas);
    return sh.Cy ? sh.C() : 0;
}

template <typename BondT, bool ALWAYS, bool RARE, bool HB, bool CLUSTER, bool YSPLIT>
static cudaError_t launch_small_kernel(const SmallArgs &a, int C, unsigned threads, size_t smem, cudaStream_t st)
{
    auto kern = k_sweep_small<BondT, ALWAYS, RARE, HB, CLUSTER, YSPLIT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (C > 8 && (e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1)) != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)C);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = CLUSTER ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, a);
}

template <typename BondT, bool CLUSTER, bool YSPLIT>
static cudaError_t launch_small_typed(ea_sim *s, const SmallArgs &a, int C, unsigned threads, size_t smem, cudaStream_t st)
{
    const Thresholds &th = s->th;
    if (s->dynamics == EA_DYN_HEATBATH) return launch_small_kernel<BondT, false, false, true, CLUSTER, YSPLIT>(a, C, threads, smem, st);
    const bool always = th.always[0] | th.always[1] | th.always[2];
    // The warp-level branch around the energy-raising levels (RARE, as in the persistent L = 128 kernel) saves alu issue
    // slots, which only bind with four warps per sub-partition (L = 32: 0.65 against 0.70 us); with one or two the
    // branch-free predicated levels schedule better (L = 8: 0.18 against 0.27 us, L = 16: 0.30 against 0.35, L = 24: 0.44 / 0.47)
    // -- unless many sims share the SMs (ea_set_concurrency_hint), which makes the issue slots bind again (64 points of
    // L = 16: 1.40 against 1.62 us per sweep of all of them).
    const bool shared = (long)s->n_concurrent * C > s->n_sm;
    const bool rare = (threads > 256 || shared) && !always && th.thr[2] < 0x04000000u;
    return always ? launch_small_kernel<BondT, true, false, false, CLUSTER, YSPLIT>(a, C, threads, smem, st)
           : rare ? launch_small_kernel<BondT, false, true, false, CLUSTER, YSPLIT>(a, C, threads, smem, st)
                  : launch_small_kernel<BondT, false, false, false, CLUSTER, YSPLIT>(a, C, threads, smem, st);
}

bool small_supported(const ea_sim *s, std::string *why)
{
    auto no = [&](const char *msg) { if (why) *why = msg; return false; };
    const SmallShape sh = small_shape(s->lat.L, s->n_replicas);
    const int C = sh.Cy ? sh.C() : 0;
    if (!C) return no("small-lattice kernel: L must be a multiple of 4 whose blocks fit one thread-block cluster (L <= 32)");
    const int Ly = s->lat.L / sh.Cy, Lz = s->lat.L / sh.Cz;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) return no("small-lattice kernel: cudaGetDeviceProperties failed");
    if (prop.major < 9 && C > 1) return no("small-lattice kernel: the device has no thread-block clusters");
    const size_t smem = small_smem_bytes(s->lat.L, Ly, Lz, s->bond_bytes());
    if (prop.sharedMemPerBlockOptin < smem) return no("small-lattice kernel: the device has too little shared memory per CTA");
    if (C > 1) { // can the device co-schedule one cluster of this shape at all (MIG slices, small parts)?
        auto kern = k_sweep_small<uint32_t, false, true, false, true, false>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            (C > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess))
            return no("small-lattice kernel: the device rejects the cluster configuration");
        const unsigned pairs = (unsigned)((size_t)(s->lat.L / 4) * Ly * Lz);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)C);
        cfg.blockDim = dim3((pairs + 31) / 32 * 32);
        cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)C;
        attr[0].val.clusterDim.y = attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        int n_clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&n_clusters, kern, &cfg) != cudaSuccess || n_clusters < 1) {
            cudaGetLastError(); // clear
            return no("small-lattice kernel: the device cannot co-schedule a thread-block cluster of this size");
        }
    }
    return true;
}

// n sweeps starting at sweep index t0, one launch.  Asynchronous.
cudaError_t launch_sweeps_small(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st)
{
    const int L = s->lat.L;
    const SmallShape sh = small_shape(L, s->n_replicas);
    if (!sh.Cy) return cudaErrorInvalidConfiguration;
    const int C = sh.C();
    SmallArgs a;
    a.spins = s->spins;
    a.bonds = s->bonds;
    a.seed = s->seed;
    a.t0 = t0;
    a.n_half = 2 * n;
    a.L = L;
    a.Ly = L / sh.Cy;
    a.Lz = L / sh.Cz;
    a.Cy = sh.Cy;
    a.Cz = sh.Cz;
    a.th = s->th;
    const unsigned pairs = (unsigned)((size_t)(L / 4) * a.Ly * a.Lz), threads = (pairs + 31) / 32 * 32;
    const size_t smem = small_smem_bytes(L, a.Ly, a.Lz, s->bond_bytes());
    cudaError_t e;
    if (sh.Cy > 1)
        e = s->n_replicas == 2 ? launch_small_typed<uint32_t, true, true>(s, a, C, threads, smem, st)
                               : launch_small_typed<uint64_t, true, true>(s, a, C, threads, smem, st);
    else if (C > 1)
        e = s->n_replicas == 2 ? launch_small_typed<uint32_t, true, false>(s, a, C, threads, smem, st)
                               : launch_small_typed<uint64_t, true, false>(s, a, C, threads, smem, st);
    else
        e = s->n_replicas == 2 ? launch_small_typed<uint32_t, false, false>(s, a, C, threads, smem, st)
                               : launch_small_typed<uint64_t, false, false>(s, a, C, threads, smem, st);
    if (e == cudaSuccess) s->count_launch();
    return e;
}

} // namespace ea

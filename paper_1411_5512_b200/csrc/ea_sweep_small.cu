// ea_sweep_small.cu -- SMALL: the whole lattice in shared memory for the n sweeps of one ea_sweep(n) call, for the
// small lattices of the paper's scans (L = 8 .. 32: PAPER.md:134 and BASELINE configs 1-2), where a kernel launch
// per colour costs far more than the half-sweep itself.
//
// Same update and the same stream contract as every other variant, hence bit-identical.  The lattice is cut into C
// slabs of L x L x (L / C) sites along z, one CTA per slab:
//   * C = 1 (L <= 16): one CTA, the colour barrier is __syncthreads();
//   * C = 2 .. 16 (L = 32: 16 CTAs of 2 planes): one thread-block CLUSTER; a slab's boundary planes are read straight out
//     of the neighbouring CTA's shared memory (distributed shared memory, ld.shared::cluster) and the colour barrier is
//     the cluster barrier (barrier.cluster.arrive.release / wait.acquire) -- no global memory traffic between sweeps.
// Spins AND bond words live in shared memory; global memory is read once at the start and written once at the end.
// A thread owns one pair of x-adjacent same-colour sites of each colour (one Philox block per pair and sweep, C-A7).
#include <string.h>

#include "ea_internal.h"
#include "ea_sweep_common.cuh"

namespace ea {

struct SmallArgs {
    uint64_t *spins;     // [2][Nh]
    const void *bonds;   // BondT [2][3][Nh]
    uint64_t seed;
    uint64_t t0;         // first sweep index
    uint32_t n_half;     // half-sweeps to run
    int L, Lz;           // side; planes per CTA (L / cluster size)
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
__device__ __forceinline__ ulonglong2 ld_cluster128(uint32_t addr)
{
    ulonglong2 v;
    asm volatile("ld.shared::cluster.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
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
__device__ __forceinline__ void lds_bond(uint32_t addr, uint32_t &v) { asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); }
__device__ __forceinline__ void lds_bond(uint32_t addr, uint64_t &v) { asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(addr) : "memory"); }
__device__ __forceinline__ void sts_v2u64(uint32_t addr, ulonglong2 v)
{
    asm volatile("st.shared.v2.u64 [%0], {%1, %2};" ::"r"(addr), "l"(v.x), "l"(v.y) : "memory");
}

// Shared-memory addresses of everything one half-sweep of colour c touches for the thread's pair
struct SmallAddr {
    uint32_t own, x0, x1, x2, pm, pp, zm, zp;   // spins: own pair; the row's three other-colour words; y -/+ and z -/+ pairs
    uint32_t jx, jy, jz, bl0, bl1, by, bz;      // bonds: forward pairs of the own sites; +x bonds of the left neighbours; backward y, z pairs
};

__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// (A neighbour-only barrier -- remote mbarrier arrives on the two z-neighbouring CTAs, release / acquire at cluster scope --
// was measured SLOWER than the hardware cluster barrier: L = 16 on 4 CTAs 0.81 against 0.67 us per half-sweep, L = 32 on 16
// CTAs 1.32 against 1.15.  The hardware barrier is split instead: arrive, draw the next random numbers, wait.)

// Shared memory of one CTA (nh = L L Lz / 2 words per colour of the slab, pw = L L / 2 words per colour and plane):
//   spins  uint64 [2][nh]
//   bonds  BondT  [2][3][nh]
//   bzh    BondT  [2][pw]      z-bonds of the plane below the slab (the backward z bonds of the slab's first plane)
template <typename BondT, bool ALWAYS, bool RARE, bool HB, bool CLUSTER>
__global__ void __launch_bounds__(512, 1) k_sweep_small(const SmallArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_small[];
    const unsigned L = a.L, Lh = L / 2, Lz = a.Lz, hp = Lh / 2; // hp: pairs per row
    const unsigned pw = L * Lh, nh = pw * Lz, Nh = pw * L;
    const unsigned rank = CLUSTER ? cluster_ctarank() : 0, C = CLUSTER ? cluster_nctarank() : 1;
    const unsigned z0 = rank * Lz;
    uint64_t *spins_s = (uint64_t *)smem_small;
    BondT *bonds_s = (BondT *)(spins_s + 2 * nh);
    BondT *bzh_s = bonds_s + 6 * nh;
    const BondT *__restrict__ gb = (const BondT *)a.bonds;
    const unsigned tid = threadIdx.x, nthr = blockDim.x;

    // ---- prologue: the slab (contiguous in every colour / direction plane of the global arrays) ------------------
    for (unsigned v = tid; v < 2 * nh; v += nthr) {
        const unsigned c = v / nh, i = v % nh;
        spins_s[v] = a.spins[(size_t)c * Nh + (size_t)pw * z0 + i];
    }
    for (unsigned v = tid; v < 6 * nh; v += nthr) {
        const unsigned cd = v / nh, i = v % nh;
        bonds_s[v] = gb[(size_t)cd * Nh + (size_t)pw * z0 + i];
    }
    {
        const unsigned zb = (z0 + L - 1) % L;
        for (unsigned v = tid; v < 2 * pw; v += nthr) {
            const unsigned c = v / pw, i = v % pw;
            bzh_s[v] = gb[(size_t)(c * 3 + 2) * Nh + (size_t)pw * zb + i];
        }
    }

    // ---- the thread's pair: (p, y, zl) -> compact words 2p, 2p + 1 of row (y, zl), both colours -------------------
    const unsigned n_pairs = hp * L * Lz;
    const bool active = tid < n_pairs;
    const unsigned p = tid % hp, y = (tid / hp) % L, zl = active ? tid / (hp * L) : 0;
    const unsigned ym = y == 0 ? L - 1 : y - 1, yp = y + 1 == L ? 0 : y + 1;
    const unsigned i0 = Lh * (y + L * zl) + 2 * p;          // own words (and the other colour's words of the same position)
    const unsigned rowb = Lh * (y + L * zl);
    const unsigned i_ym = Lh * (ym + L * zl) + 2 * p, i_yp = Lh * (yp + L * zl) + 2 * p;
    // z neighbours: inside the slab, or the facing plane of the neighbouring CTA (C = 1: the slab wraps onto itself)
    const bool lo_edge = zl == 0, hi_edge = zl + 1 == Lz;
    const unsigned i_zm = Lh * (y + L * (lo_edge ? Lz - 1 : zl - 1)) + 2 * p;
    const unsigned i_zp = Lh * (y + L * (hi_edge ? 0 : zl + 1)) + 2 * p;
    const uint32_t spins_a = small_smem_u32(spins_s);
    uint32_t base_zm = spins_a, base_zp = spins_a; // shared::cluster addresses of the spin array that holds the z -/+ neighbour
    if (CLUSTER) {
        base_zm = mapa_u32(spins_a, lo_edge ? (rank + C - 1) % C : rank);
        base_zp = mapa_u32(spins_a, hi_edge ? (rank + 1) % C : rank);
    }
    const unsigned zg = z0 + zl;
    const uint32_t site_row = L * (y + L * zg);

    // per colour c: x-phase S = (c ^ y ^ z) & 1; the three other-colour words of the row next to the pair are compact
    // q, q + 1, q + 2 with q = 2p - 1 + S (periodic)
    unsigned Sc[2];
    SmallAddr A[2];
    const uint32_t bonds_a = small_smem_u32(bonds_s), bzh_a = small_smem_u32(bzh_s);
    constexpr unsigned BS = sizeof(BondT);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        Sc[c] = (c ^ y ^ zg) & 1u;
        const unsigned q0 = (2 * p + Sc[c] + Lh - 1) % Lh, q1 = (q0 + 1) % Lh, q2 = (q1 + 1) % Lh;
        const unsigned own_w = c * nh, oth_w = (1 - c) * nh;
        A[c].own = spins_a + (own_w + i0) * 8;
        A[c].x0 = spins_a + (oth_w + rowb + q0) * 8;
        A[c].x1 = spins_a + (oth_w + rowb + q1) * 8;
        A[c].x2 = spins_a + (oth_w + rowb + q2) * 8;
        A[c].pm = spins_a + (oth_w + i_ym) * 8;
        A[c].pp = spins_a + (oth_w + i_yp) * 8;
        A[c].zm = base_zm + (oth_w + i_zm) * 8;
        A[c].zp = base_zp + (oth_w + i_zp) * 8;
        const unsigned jc_w = c * 3 * nh, jo_w = (1 - c) * 3 * nh;
        A[c].jx = bonds_a + (jc_w + i0) * BS;
        A[c].jy = bonds_a + (jc_w + nh + i0) * BS;
        A[c].jz = bonds_a + (jc_w + 2 * nh + i0) * BS;
        A[c].bl0 = bonds_a + (jo_w + rowb + q0) * BS;
        A[c].bl1 = bonds_a + (jo_w + rowb + q1) * BS;
        A[c].by = bonds_a + (jo_w + nh + i_ym) * BS;
        A[c].bz = lo_edge ? bzh_a + ((1 - c) * pw + Lh * y + 2 * p) * BS : bonds_a + (jo_w + 2 * nh + i_zm) * BS;
    }
    const uint32_t site0 = site_row + 4 * p + Sc[0], site1 = site_row + 4 * p + Sc[1]; // first site of the pair, colour 0 / 1

    auto half_sweep = [&](const SmallAddr &ad, const uint4 r) {
        const uint64_t X0 = lds_u64(ad.x0), X1 = lds_u64(ad.x1), X2 = lds_u64(ad.x2);
        const ulonglong2 own = lds_v2u64(ad.own), Pm = lds_v2u64(ad.pm), Pp = lds_v2u64(ad.pp);
        const ulonglong2 Zm = CLUSTER ? ld_cluster128(ad.zm) : lds_v2u64(ad.zm);
        const ulonglong2 Zp = CLUSTER ? ld_cluster128(ad.zp) : lds_v2u64(ad.zp);
        BondT jxA, jxB, jyA, jyB, jzA, jzB, bl0, bl1, byA, byB, bzA, bzB;
        lds_bond(ad.jx, jxA); lds_bond(ad.jx + BS, jxB);
        lds_bond(ad.jy, jyA); lds_bond(ad.jy + BS, jyB);
        lds_bond(ad.jz, jzA); lds_bond(ad.jz + BS, jzB);
        lds_bond(ad.bl0, bl0); lds_bond(ad.bl1, bl1);
        lds_bond(ad.by, byA); lds_bond(ad.by + BS, byB);
        lds_bond(ad.bz, bzA); lds_bond(ad.bz + BS, bzB);
        ulonglong2 out;
        out.x = metropolis_word<BondT, ALWAYS, RARE, HB>(own.x, X1, X0, Pp.x, Pm.x, Zp.x, Zm.x, jxA, bl0, jyA, byA, jzA, bzA, r.x, r.y, a.th);
        out.y = metropolis_word<BondT, ALWAYS, RARE, HB>(own.y, X2, X1, Pp.y, Pm.y, Zp.y, Zm.y, jxB, bl1, jyB, byB, jzB, bzB, r.z, r.w, a.th);
        sts_v2u64(ad.own, out);
    };

    // end of a half-sweep: arrive at the colour barrier, draw the next random numbers meanwhile, wait
    auto barrier_begin = [&]() {
        if (CLUSTER) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    };
    auto barrier_end = [&]() {
        if (CLUSTER) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
        else __syncthreads();
    };

    SweepRng g = make_sweep_rng(a.seed, a.t0, 0);
    // the random numbers do not depend on the spins: those of the next half-sweep are drawn while the barrier completes
    uint4 r = sweep_random4(g, site0);
    if (CLUSTER) cluster_barrier(); else __syncthreads(); // every CTA of the cluster has its slab in place

    for (uint32_t sw = 0; sw < a.n_half / 2; ++sw) { // n_half is even: colour 0 then colour 1 of sweep t0 + sw
        if (active) half_sweep(A[0], r);
        barrier_begin();
        sweep_rng_set_time(g, a.t0 + sw, 1u);
        r = sweep_random4(g, site1);
        barrier_end();
        if (active) half_sweep(A[1], r);
        barrier_begin();
        sweep_rng_set_time(g, a.t0 + sw + 1, 0u);
        r = sweep_random4(g, site0);
        barrier_end();
    }
    if (CLUSTER) cluster_barrier(); // nobody leaves while a neighbour may still read its shared memory

    // ---- epilogue: the slab back to global ---------------------------------------------------------------------------
    for (unsigned v = tid; v < 2 * nh; v += nthr) {
        const unsigned c = v / nh, i = v % nh;
        a.spins[(size_t)c * Nh + (size_t)pw * z0 + i] = spins_s[v];
    }
}

// ---------------------------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------------------------
static size_t small_smem_bytes(int L, int Lz, int bond_bytes)
{
    const size_t pw = (size_t)L * L / 2, nh = pw * Lz;
    return 2 * nh * 8 + 6 * nh * bond_bytes + 2 * pw * bond_bytes;
}

// Cluster size C (1, 2, 4, 8, 16; L % C == 0) for a lattice of side L: every slab must fit one CTA (at most 512 pairs =
// threads, and the shared memory of one SM); among those the one with the smallest estimated half-sweep time -- warps per
// sub-partition x ~300 clocks per pair, plus ~40 clocks for __syncthreads() or ~450 for the cluster barrier (measured:
// L = 16 on one CTA 1.93 us, L = 32 on 8 CTAs 1.84 us).  0 if there is none.
int small_cluster_size(int L, int n_replicas)
{
    if (L < 4 || L % 4 || L > 64) return 0;
    const int bond_bytes = n_replicas == 2 ? 4 : 8;
    int best = 0;
    long best_cost = 0;
    for (int C = 1; C <= 16; C *= 2) {
        if (L % C) continue;
        const int Lz = L / C;
        const long pairs = (long)L * L * Lz / 4;
        if (pairs > 512 || small_smem_bytes(L, Lz, bond_bytes) > 200 * 1024) continue;
        const long cost = (pairs + 127) / 128 * 300 + (C > 1 ? 450 : 40);
        if (!best || cost < best_cost) { best = C; best_cost = cost; }
    }
    return best;
}

template <typename BondT, bool ALWAYS, bool RARE, bool HB, bool CLUSTER>
static cudaError_t launch_small_kernel(const SmallArgs &a, int C, unsigned threads, size_t smem, cudaStream_t st)
{
    auto kern = k_sweep_small<BondT, ALWAYS, RARE, HB, CLUSTER>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (C > 8 && (e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1)) != cudaSuccess) return e;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
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

template <typename BondT, bool CLUSTER>
static cudaError_t launch_small_typed(ea_sim *s, const SmallArgs &a, int C, unsigned threads, size_t smem, cudaStream_t st)
{
    const Thresholds &th = s->th;
    if (s->dynamics == EA_DYN_HEATBATH) return launch_small_kernel<BondT, false, false, true, CLUSTER>(a, C, threads, smem, st);
    const bool always = th.always[0] | th.always[1] | th.always[2];
    const bool rare = !always && th.thr[2] < 0x04000000u; // as in the persistent L = 128 kernel
    return always ? launch_small_kernel<BondT, true, false, false, CLUSTER>(a, C, threads, smem, st)
           : rare ? launch_small_kernel<BondT, false, true, false, CLUSTER>(a, C, threads, smem, st)
                  : launch_small_kernel<BondT, false, false, false, CLUSTER>(a, C, threads, smem, st);
}

bool small_supported(const ea_sim *s, std::string *why)
{
    auto no = [&](const char *msg) { if (why) *why = msg; return false; };
    const int C = small_cluster_size(s->lat.L, s->n_replicas);
    if (!C) return no("small-lattice kernel: L must be a multiple of 4 whose slabs fit one thread-block cluster (L <= 32)");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) return no("small-lattice kernel: cudaGetDeviceProperties failed");
    if (prop.major < 9 && C > 1) return no("small-lattice kernel: the device has no thread-block clusters");
    const size_t smem = small_smem_bytes(s->lat.L, s->lat.L / C, s->bond_bytes());
    if (prop.sharedMemPerBlockOptin < smem) return no("small-lattice kernel: the device has too little shared memory per CTA");
    if (C > 1) { // can the device co-schedule one cluster of this shape at all (MIG slices, small parts)?
        auto kern = k_sweep_small<uint32_t, false, true, false, true>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            (C > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess))
            return no("small-lattice kernel: the device rejects the cluster configuration");
        const unsigned pairs = (unsigned)((size_t)s->lat.L * s->lat.L * (s->lat.L / C) / 4);
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
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
    const int L = s->lat.L, C = small_cluster_size(L, s->n_replicas);
    if (!C) return cudaErrorInvalidConfiguration;
    SmallArgs a;
    a.spins = s->spins;
    a.bonds = s->bonds;
    a.seed = s->seed;
    a.t0 = t0;
    a.n_half = 2 * n;
    a.L = L;
    a.Lz = L / C;
    a.th = s->th;
    const unsigned pairs = (unsigned)((size_t)L * L * a.Lz / 4), threads = (pairs + 31) / 32 * 32;
    const size_t smem = small_smem_bytes(L, a.Lz, s->bond_bytes());
    cudaError_t e;
    if (C > 1)
        e = s->n_replicas == 2 ? launch_small_typed<uint32_t, true>(s, a, C, threads, smem, st)
                               : launch_small_typed<uint64_t, true>(s, a, C, threads, smem, st);
    else
        e = s->n_replicas == 2 ? launch_small_typed<uint32_t, false>(s, a, C, threads, smem, st)
                               : launch_small_typed<uint64_t, false>(s, a, C, threads, smem, st);
    if (e == cudaSuccess) s->count_launch();
    return e;
}

} // namespace ea

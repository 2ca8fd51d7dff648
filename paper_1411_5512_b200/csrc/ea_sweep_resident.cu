// ea_sweep_resident.cu -- RESIDENT: a persistent half-sweep kernel for L = 128 that keeps the whole spin
// lattice in shared memory for the n sweeps of one ea_sweep(n) call.
//
// Same update as every other variant (Eq. 9; checkerboard order PAPER.md:80-86) and the same
// stream contract, hence bit-identical results.  What changes is where the colour barrier ("each
// half-step is performed in its own CUDA kernel call to ensure global synchronization") comes from:
//
//   * the y-z plane of rows is cut into (L/TY) x (L/TZ) tiles, one CTA per tile, one CTA per SM (cooperative
//     launch: all CTAs are co-resident).  A CTA holds both colours of its TY x TZ rows plus a one-row halo ring
//     in shared memory: 2 x (TZ+2) x (TY+2) x 512 B = 180 KB for TY = 16, TZ = 8 (128 CTAs).
//   * a half-step updates one colour of the tile from shared memory; only the bond words stream in (from L2:
//     bonds never change).  Boundary rows are updated first and also stored to the global spin array; a
//     producer warp then publishes "step h done" (fence + flag), waits for the same flag of the four
//     neighbouring tiles and pulls their fresh boundary rows into the halo ring with 1-D bulk TMA copies,
//     while the compute warps update the interior rows.  The colour barrier is therefore a neighbour-only
//     dependency whose latency is hidden behind the interior update -- no grid-wide barrier, no relaunch.
//   * global memory always holds the current boundary rows; interior rows are written back once at the end,
//     so after the launch the global array is the full state at time t0 + n.
#include <cooperative_groups.h>

#include "ea_internal.h"
#include "ea_sweep_common.cuh"

namespace ea {

struct ResidentArgs {
    uint64_t *spins;     // [2][Nh]
    const void *bonds;   // BondT [2][3][Nh]
    uint64_t seed;
    uint64_t t0;         // first sweep index
    uint32_t n_half;     // half-steps to run (2 per sweep)
    uint32_t epoch0;     // flag value before this launch; step h publishes epoch0 + h + 1
    unsigned *flags;     // [G][32]: one 128-byte line per CTA
    unsigned *abort_flag;// set by any CTA whose wait timed out; everybody then leaves
    Thresholds th;
};

template <int L_, int TY_, int TZ_> struct ResidentGeom {
    static constexpr int L = L_, TY = TY_, TZ = TZ_;
    static constexpr int Lh = L / 2;                 // words per colour row
    static constexpr int NTY = L / TY, NTZ = L / TZ; // tiles along y, z
    static constexpr int G = NTY * NTZ;              // CTAs
    static constexpr int ROWS = TY * TZ;             // rows updated per CTA per half-step
    static constexpr int HY = TY + 2, HZ = TZ + 2;   // with halo ring
    static constexpr int CW = 16;                    // compute warps
    static constexpr int THREADS = (CW + 1) * 32;    // + one producer warp
    static constexpr int NB = ROWS - (TY - 2) * (TZ - 2); // boundary rows
    static constexpr unsigned HALO_BYTES = (2 * TY + 2 * TZ) * Lh * 8;
    static constexpr size_t SPIN_BYTES = (size_t)2 * HZ * HY * Lh * 8;
    static constexpr size_t SMEM_BYTES = SPIN_BYTES + 16 /*mbarrier*/ + ROWS * 4 /*row table*/;
    static_assert(Lh == 64, "a warp covers one colour row with two words per lane");
    static_assert(ROWS % CW == 0, "equal number of rows per compute warp");
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, unsigned parity)
{
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(parity)
                 : "memory");
    return ok != 0;
}
// 1-D bulk copy global -> shared (TMA unit, async proxy); completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned *p, unsigned v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

enum { BAR_BOUNDARY = 1, BAR_STEP = 2 };
constexpr unsigned long long RESIDENT_TIMEOUT_NS = 2000000000ull; // a neighbour that never shows up: give up after 2 s

template <typename BondT> struct RowBonds { typename Pair<BondT>::type jx, jy, jz, bx, by, bz; };

template <typename G, typename BondT>
__device__ __forceinline__ RowBonds<BondT> load_row_bonds(const BondT *__restrict__ Jc, const BondT *__restrict__ Jo,
                                                          unsigned y, unsigned z, unsigned k)
{
    constexpr unsigned Lh = G::Lh, L = G::L, Nh = (unsigned)L * L * L / 2;
    const unsigned row = Lh * (y + L * z) + 2 * k;
    const unsigned rowym = Lh * (((y - 1) & (L - 1)) + L * z) + 2 * k;
    const unsigned rowzm = Lh * (y + L * ((z - 1) & (L - 1))) + 2 * k;
    RowBonds<BondT> b;
    b.jx = ldg_pair<BondT>(Jc + row);
    b.jy = ldg_pair<BondT>(Jc + Nh + row);
    b.jz = ldg_pair<BondT>(Jc + 2 * Nh + row);
    b.bx = ldg_pair<BondT>(Jo + row);
    b.by = ldg_pair<BondT>(Jo + Nh + rowym);
    b.bz = ldg_pair<BondT>(Jo + 2 * Nh + rowzm);
    return b;
}

template <typename G, typename BondT, bool ALWAYS>
__global__ void __launch_bounds__(G::THREADS, 1) k_sweep_resident(const ResidentArgs a)
{
    constexpr int L = G::L, Lh = G::Lh, TY = G::TY, TZ = G::TZ, HY = G::HY, HZ = G::HZ, CW = G::CW, ROWS = G::ROWS;
    constexpr unsigned Nh = (unsigned)L * L * L / 2;
    constexpr int RPW = ROWS / CW; // rows per compute warp per half-step
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *tile = (uint64_t *)smem_raw;                          // [2][HZ][HY][Lh]
    uint64_t *halo_bar = (uint64_t *)(smem_raw + G::SPIN_BYTES);    // mbarrier: halo of the next step has landed
    uint32_t *rowtab = (uint32_t *)(smem_raw + G::SPIN_BYTES + 16); // [ROWS]: yy | zz << 8, boundary rows first

    const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned b = blockIdx.x, ty = b % G::NTY, tz = b / G::NTY;
    const unsigned y0 = ty * TY, z0 = tz * TZ;
    auto tile_at = [&](int c, int zz, int yy) -> uint64_t * { return tile + ((size_t)(c * HZ + zz) * HY + yy) * Lh; };

    // ---- prologue: row table, barrier, tile + halo ring of both colours from global -------------------
    if (tid < (unsigned)ROWS) {
        const int yy = 1 + (int)tid % TY, zz = 1 + (int)tid / TY;
        const bool isB = yy == 1 || yy == TY || zz == 1 || zz == TZ;
        int before_same = 0;
        for (int j = 0; j < (int)tid; ++j) {
            const int y2 = 1 + j % TY, z2 = 1 + j / TY;
            const bool b2 = y2 == 1 || y2 == TY || z2 == 1 || z2 == TZ;
            before_same += (b2 == isB);
        }
        rowtab[isB ? before_same : G::NB + before_same] = (uint32_t)yy | ((uint32_t)zz << 8);
    }
    if (tid == 0) {
        mbar_init(halo_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (unsigned v = tid; v < 2u * HZ * HY * (Lh / 2); v += G::THREADS) {
        const unsigned w2 = v % (Lh / 2), r = v / (Lh / 2);
        const unsigned yy = r % HY, zz = (r / HY) % HZ, c = r / (HY * HZ);
        const unsigned y = (y0 + yy - 1) & (L - 1), z = (z0 + zz - 1) & (L - 1);
        const ulonglong2 val = *(const ulonglong2 *)(a.spins + (size_t)c * Nh + Lh * (y + L * z) + 2 * w2);
        *(ulonglong2 *)(tile_at(c, zz, yy) + 2 * w2) = val;
    }
    __syncthreads();

    const BondT *__restrict__ bonds = (const BondT *)a.bonds;

    if (warp == (unsigned)CW) {
        // ---- producer warp: publish our boundary rows, fetch the neighbours' --------------------------
        const unsigned nb_tile = lane == 0   ? ((ty + 1) % G::NTY) + G::NTY * tz
                                 : lane == 1 ? ((ty + G::NTY - 1) % G::NTY) + G::NTY * tz
                                 : lane == 2 ? ty + G::NTY * ((tz + 1) % G::NTZ)
                                             : ty + G::NTY * ((tz + G::NTZ - 1) % G::NTZ);
        for (uint32_t h = 0; h < a.n_half; ++h) {
            const int c = h & 1;
            named_bar_sync(BAR_BOUNDARY, G::THREADS); // boundary rows of step h are in smem and in global
            const unsigned epoch = a.epoch0 + h + 1;
            if (lane == 0) {
                __threadfence();
                st_release_gpu(a.flags + b * 32, epoch);
            }
            if (h + 1 == a.n_half) break;
            bool ok = true;
            if (lane < 4) {
                const unsigned *f = a.flags + nb_tile * 32;
                const unsigned long long t_start = globaltimer_ns();
                unsigned spins = 0;
                while ((int)(ld_acquire_gpu(f) - epoch) < 0) {
                    if ((++spins & 63u) == 0) {
                        if (*(volatile unsigned *)a.abort_flag || globaltimer_ns() - t_start > RESIDENT_TIMEOUT_NS) {
                            ok = false;
                            break;
                        }
                    }
                }
            }
            ok = __all_sync(0xffffffffu, ok);
            if (!ok) {
                if (lane == 0) atomicExch(a.abort_flag, 1u);
                // leave the halo stale; everybody notices the abort flag below and the host reports the error
            }
            if (lane == 0) {
                asm volatile("fence.proxy.async;" ::: "memory");
                mbar_arrive_expect_tx(halo_bar, G::HALO_BYTES);
                const uint64_t *src = a.spins + (size_t)c * Nh;
                const unsigned zlo = (z0 - 1) & (L - 1), zhi = (z0 + TZ) & (L - 1);
                const unsigned ylo = (y0 - 1) & (L - 1), yhi = (y0 + TY) & (L - 1);
                bulk_g2s(tile_at(c, 0, 1), src + Lh * (y0 + L * zlo), TY * Lh * 8, halo_bar);
                bulk_g2s(tile_at(c, HZ - 1, 1), src + Lh * (y0 + L * zhi), TY * Lh * 8, halo_bar);
                for (int zz = 1; zz <= TZ; ++zz) {
                    const unsigned z = z0 + zz - 1;
                    bulk_g2s(tile_at(c, zz, 0), src + Lh * (ylo + L * z), Lh * 8, halo_bar);
                    bulk_g2s(tile_at(c, zz, HY - 1), src + Lh * (yhi + L * z), Lh * 8, halo_bar);
                }
            }
        }
    } else {
        // ---- compute warps -----------------------------------------------------------------------------
        const unsigned k = lane;
        const int lane_m = (int)((k - 1) & 31), lane_p = (int)((k + 1) & 31);
        int n_bnd = 0; // boundary rows of this warp: indices warp + CW*i < NB
        for (int i = 0; i < RPW; ++i) n_bnd += ((int)warp + CW * i < G::NB);
        uint32_t rt[RPW];
#pragma unroll
        for (int i = 0; i < RPW; ++i) rt[i] = rowtab[warp + CW * i];

        RowBonds<BondT> nxt; // software pipeline: the bond words of the next row are in flight during this row
        {
            const unsigned yy = rt[0] & 0xff, zz = rt[0] >> 8;
            nxt = load_row_bonds<G, BondT>(bonds, bonds + (size_t)3 * Nh, y0 + yy - 1, z0 + zz - 1, k);
        }
        for (uint32_t h = 0; h < a.n_half; ++h) {
            const int c = h & 1;
            const SweepRng g = make_sweep_rng(a.seed, a.t0 + (h >> 1), (uint32_t)c);
            const BondT *__restrict__ Jc = bonds + (size_t)c * 3 * Nh;
            const BondT *__restrict__ Jo = bonds + (size_t)(1 - c) * 3 * Nh;
            uint64_t *gown = a.spins + (size_t)c * Nh;
            if (h > 0) { // halo of colour 1-c, pulled in during step h-1
                const unsigned parity = (h - 1) & 1;
                while (!mbar_try_wait(halo_bar, parity)) { } // always completes: the producer arms it even on abort
            }
            if (n_bnd == 0) named_bar_arrive(BAR_BOUNDARY, G::THREADS);
#pragma unroll
            for (int i = 0; i < RPW; ++i) {
                const unsigned yy = rt[i] & 0xff, zz = rt[i] >> 8;
                const unsigned y = y0 + yy - 1, z = z0 + zz - 1;
                const RowBonds<BondT> cur = nxt;
                { // prefetch the next row's bonds (next half-step's first row at the end of this one)
                    const uint32_t e = rt[(i + 1) % RPW];
                    const unsigned yn = y0 + (e & 0xff) - 1, zn = z0 + (e >> 8) - 1;
                    if (i + 1 < RPW) nxt = load_row_bonds<G, BondT>(Jc, Jo, yn, zn, k);
                    else nxt = load_row_bonds<G, BondT>(Jo, Jc, yn, zn, k); // colours swap roles next step
                }
                uint64_t *own_row = tile_at(c, zz, yy) + 2 * k;
                const ulonglong2 own = *(const ulonglong2 *)own_row;
                const ulonglong2 P0 = *(const ulonglong2 *)(tile_at(1 - c, zz, yy) + 2 * k);
                const ulonglong2 Pm = *(const ulonglong2 *)(tile_at(1 - c, zz, yy - 1) + 2 * k);
                const ulonglong2 Pp = *(const ulonglong2 *)(tile_at(1 - c, zz, yy + 1) + 2 * k);
                const ulonglong2 Zm = *(const ulonglong2 *)(tile_at(1 - c, zz - 1, yy) + 2 * k);
                const ulonglong2 Zp = *(const ulonglong2 *)(tile_at(1 - c, zz + 1, yy) + 2 * k);
                const unsigned s = ((unsigned)c ^ (y + z)) & 1u;
                const uint32_t site0 = 4 * k + s + L * (y + L * z);
                ulonglong2 out;
                if (s == 0)
                    out = update_pair<0, BondT, ALWAYS>(own, P0, Pm, Pp, Zm, Zp, cur.jx, cur.jy, cur.jz, cur.bx, cur.by,
                                                       cur.bz, site0, g, a.th, lane_m, lane_p);
                else
                    out = update_pair<1, BondT, ALWAYS>(own, P0, Pm, Pp, Zm, Zp, cur.jx, cur.jy, cur.jz, cur.bx, cur.by,
                                                       cur.bz, site0, g, a.th, lane_m, lane_p);
                *(ulonglong2 *)own_row = out;
                if (i < n_bnd) {
                    *(ulonglong2 *)(gown + Lh * (y + L * z) + 2 * k) = out;
                    if (i == n_bnd - 1) named_bar_arrive(BAR_BOUNDARY, G::THREADS);
                }
            }
            named_bar_sync(BAR_STEP, CW * 32); // colour c of the tile is complete before anyone reads it
        }
        // ---- epilogue: interior rows were never stored; write them back (boundary rows are current) ----
#pragma unroll
        for (int i = 0; i < RPW; ++i) {
            if (i < n_bnd) continue;
            const unsigned yy = rt[i] & 0xff, zz = rt[i] >> 8;
            const unsigned y = y0 + yy - 1, z = z0 + zz - 1;
#pragma unroll
            for (int c = 0; c < 2; ++c)
                *(ulonglong2 *)(a.spins + (size_t)c * Nh + Lh * (y + L * z) + 2 * k) =
                    *(const ulonglong2 *)(tile_at(c, zz, yy) + 2 * k);
        }
    }
}

// ---------------------------------------------------------------------------------------------
typedef ResidentGeom<128, 16, 8> Geom128;

template <typename BondT, bool ALWAYS>
static cudaError_t launch_resident_typed(ea_sim *s, ResidentArgs &a, cudaStream_t st)
{
    auto kern = k_sweep_resident<Geom128, BondT, ALWAYS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Geom128::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    void *args[] = {&a};
    return cudaLaunchCooperativeKernel((void *)kern, dim3(Geom128::G), dim3(Geom128::THREADS), args, Geom128::SMEM_BYTES, st);
}

bool resident_supported(const ea_sim *s)
{
    if (s->lat.L != 128) return false;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) return false;
    return prop.cooperativeLaunch && prop.multiProcessorCount >= Geom128::G &&
           prop.sharedMemPerBlockOptin >= Geom128::SMEM_BYTES;
}

size_t resident_flag_bytes() { return (size_t)(Geom128::G * 32 + 32) * sizeof(unsigned); }

// n sweeps starting at sweep index t0, one launch.  Asynchronous; ea_sim::resident_epoch advances by 2n.
cudaError_t launch_sweeps_resident(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st)
{
    ResidentArgs a;
    a.spins = s->spins;
    a.bonds = s->bonds;
    a.seed = s->seed;
    a.t0 = t0;
    a.n_half = 2 * n;
    a.epoch0 = s->resident_epoch;
    a.flags = s->resident_flags;
    a.abort_flag = s->resident_flags + Geom128::G * 32;
    a.th = s->th;
    const bool always = a.th.always[0] | a.th.always[1] | a.th.always[2];
    cudaError_t e;
    if (s->n_replicas == 2)
        e = always ? launch_resident_typed<uint32_t, true>(s, a, st) : launch_resident_typed<uint32_t, false>(s, a, st);
    else
        e = always ? launch_resident_typed<uint64_t, true>(s, a, st) : launch_resident_typed<uint64_t, false>(s, a, st);
    if (e == cudaSuccess) {
        s->resident_epoch += 2 * n;
        s->count_launch();
    }
    return e;
}

} // namespace ea

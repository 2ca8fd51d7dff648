// ea_sweep.cu -- the half-sweep kernels: one Metropolis trial (Eq. 9) for every site of one
// colour, 64 samples per word, in the colour-split compact layout of ea_device.cuh.
//
// A kernel boundary is the colour barrier ("each half-step is performed in its own CUDA kernel call to
// ensure global synchronization").  All variants are bit-identical (same stream contract).
#include <cooperative_groups.h>
#include <string.h>

#include "ea_internal.h"
#include "ea_sweep_common.cuh"

namespace ea {

struct SweepArgs {
    Lattice lat;
    int colour;                 // parity of the sites updated by this launch (C-S2)
    uint64_t *own;              // spins[colour]      (read + written)
    const uint64_t *oth;        // spins[1 - colour]  (read only)
    const void *Jc;             // bonds[colour][3][Nh]     forward bonds of the updated sites
    const void *Jo;             // bonds[1 - colour][3][Nh] forward bonds of the neighbours (our backward bonds)
    uint64_t seed;
    uint64_t t;                 // sweep index, used when d_time == nullptr
    const uint64_t *d_time;     // device-resident t (CUDA-graph replays); t = *d_time + t_offset
    uint32_t t_offset;
    Thresholds th;
};

__device__ __forceinline__ uint64_t sweep_time(const SweepArgs &a)
{
    return (a.d_time ? *a.d_time : a.t) + a.t_offset;
}

// Programmatic dependent launch: consecutive half-sweep launches depend on each other completely (the colour barrier,
// PAPER.md:86), but the NEXT launch's grid can be brought onto the SMs while this one still runs: every sweep kernel lets
// its dependents launch at once and waits for its own predecessor before it reads anything the predecessor wrote.  The
// launches carry cudaLaunchAttributeProgrammaticStreamSerialization (a programmatic edge when captured into a graph).
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

template <bool POW2>
__device__ __forceinline__ void decode_row(const Lattice &lat, unsigned tid, unsigned log2W, unsigned W, unsigned &k,
                                           unsigned &y, unsigned &z)
{
    unsigned row;
    if (POW2) {
        k = tid & (W - 1);
        row = tid >> log2W;
        y = row & (lat.L - 1);
        z = row >> lat.log2L;
    } else {
        k = tid % W;
        row = tid / W;
        y = row % lat.L;
        z = row / lat.L;
    }
}

// ---------------------------------------------------------------------------------------------
// SCALAR: one site per thread, any even L >= 2 (L = 2: +x and -x neighbours are the same site,
// reached through two distinct bonds -- C-S15).
// ---------------------------------------------------------------------------------------------
template <typename BondT, bool POW2, bool ALWAYS, bool HB>
__global__ void __launch_bounds__(256) k_sweep_scalar(const SweepArgs a)
{
    pdl_launch_dependents();
    const Lattice lat = a.lat;
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= lat.Nh) return;
    unsigned xh, y, z;
    decode_row<POW2>(lat, tid, lat.log2Lh, lat.Lh, xh, y, z);
    const unsigned L = lat.L, Lh = lat.Lh;
    const unsigned s = (a.colour ^ (y + z)) & 1u;
    const unsigned yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const unsigned zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    const unsigned rowbase = Lh * (y + L * z);
    const unsigned i = rowbase + xh;
    const unsigned xo = s ? ((xh + 1 == Lh) ? 0 : xh + 1) : ((xh == 0) ? Lh - 1 : xh - 1);
    const unsigned jp = s ? rowbase + xo : i; // compact index of the +x neighbour
    const unsigned jm = s ? i : rowbase + xo; // compact index of the -x neighbour
    const unsigned iyp = Lh * (yp + L * z) + xh, iym = Lh * (ym + L * z) + xh;
    const unsigned izp = Lh * (y + L * zp) + xh, izm = Lh * (y + L * zm) + xh;

    const BondT *__restrict__ Jc = (const BondT *)a.Jc;
    const BondT *__restrict__ Jo = (const BondT *)a.Jo;
    const unsigned Nh = lat.Nh;
    const BondT j_xp = __ldg(Jc + i), j_yp = __ldg(Jc + Nh + i), j_zp = __ldg(Jc + 2 * Nh + i); // bonds never change:
    const BondT j_xm = __ldg(Jo + jm), j_ym = __ldg(Jo + Nh + iym), j_zm = __ldg(Jo + 2 * Nh + izm); // before the wait
    pdl_wait(); // the previous half-sweep is complete; spins through L2 (the read-only path may predate it)
    const uint64_t sg = a.own[i];
    const uint64_t n_xp = __ldcg(a.oth + jp), n_xm = __ldcg(a.oth + jm);
    const uint64_t n_yp = __ldcg(a.oth + iyp), n_ym = __ldcg(a.oth + iym);
    const uint64_t n_zp = __ldcg(a.oth + izp), n_zm = __ldcg(a.oth + izm);

    const SweepRng g = make_sweep_rng(a.seed, sweep_time(a), (uint32_t)a.colour);
    const uint32_t site = (2 * xh + s) + L * (y + L * z); // canonical site index
    uint32_t r_lo, r_hi;                                   // counter word 0 = the first site of the pair (xh even)
    sweep_random(g, site - 2 * (xh & 1u), xh & 1u, r_lo, r_hi);
    a.own[i] = metropolis_word<BondT, ALWAYS, false, HB>(sg, n_xp, n_xm, n_yp, n_ym, n_zp, n_zm, j_xp, j_xm, j_yp, j_ym, j_zp, j_zm,
                                      r_lo, r_hi, a.th);
}

// ---------------------------------------------------------------------------------------------
// VEC2: two x-adjacent sites of one colour per thread; every access but one neighbour word and one
// bond word per thread is a 128-bit (uint64 pairs) or 64-bit (uint32 bond pairs) vector.  L % 4 == 0.
// ---------------------------------------------------------------------------------------------

template <typename BondT, bool POW2, bool ALWAYS, bool HB>
__global__ void __launch_bounds__(256) k_sweep_vec2(const SweepArgs a)
{
    pdl_launch_dependents();
    const Lattice lat = a.lat;
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= lat.Nh / 2) return;
    const unsigned L = lat.L, Lh = lat.Lh, W = Lh >> 1;
    unsigned k, y, z;
    decode_row<POW2>(lat, tid, lat.log2Lh - 1, W, k, y, z);
    const unsigned s = (a.colour ^ (y + z)) & 1u;
    const unsigned yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const unsigned zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    const unsigned rowbase = Lh * (y + L * z);
    const unsigned i0 = rowbase + 2 * k;
    // the one word outside the aligned pair: oth[2k-1] (s = 0, the -x neighbour of word 0) or oth[2k+2] (s = 1)
    const unsigned xe = s ? ((2 * k + 2 == Lh) ? 0 : 2 * k + 2) : ((k == 0) ? Lh - 1 : 2 * k - 1);
    const unsigned ie = rowbase + xe;
    const unsigned iyp = Lh * (yp + L * z) + 2 * k, iym = Lh * (ym + L * z) + 2 * k;
    const unsigned izp = Lh * (y + L * zp) + 2 * k, izm = Lh * (y + L * zm) + 2 * k;
    const unsigned Nh = lat.Nh;
    const BondT *__restrict__ Jc = (const BondT *)a.Jc;
    const BondT *__restrict__ Jo = (const BondT *)a.Jo;

    BondT jx0, jx1, jy0, jy1, jz0, jz1, B0, B1, by0, by1, bz0, bz1; // bonds never change: loaded before the wait
    ld_pair<BondT>(Jc + i0, jx0, jx1);
    ld_pair<BondT>(Jc + Nh + i0, jy0, jy1);
    ld_pair<BondT>(Jc + 2 * Nh + i0, jz0, jz1);
    ld_pair<BondT>(Jo + i0, B0, B1);
    const BondT Jex = __ldg(Jo + ie);
    ld_pair<BondT>(Jo + Nh + iym, by0, by1);
    ld_pair<BondT>(Jo + 2 * Nh + izm, bz0, bz1);

    pdl_wait(); // the previous half-sweep is complete; spins through L2 (the read-only path may predate it)
    const ulonglong2 vs = *(const ulonglong2 *)(a.own + i0), vA = __ldcg((const ulonglong2 *)(a.oth + i0));
    const ulonglong2 vyp = __ldcg((const ulonglong2 *)(a.oth + iyp)), vym = __ldcg((const ulonglong2 *)(a.oth + iym));
    const ulonglong2 vzp = __ldcg((const ulonglong2 *)(a.oth + izp)), vzm = __ldcg((const ulonglong2 *)(a.oth + izm));
    const uint64_t ex = __ldcg(a.oth + ie);
    const uint64_t sg0 = vs.x, sg1 = vs.y, A0 = vA.x, A1 = vA.y, yp0 = vyp.x, yp1 = vyp.y, ym0 = vym.x, ym1 = vym.y;
    const uint64_t zp0 = vzp.x, zp1 = vzp.y, zm0 = vzm.x, zm1 = vzm.y;

    // (+x neighbour, -x neighbour, backward x bond) of the two words, by row phase s
    const uint64_t np0 = s ? A1 : A0, nm0 = s ? A0 : ex;
    const uint64_t np1 = s ? ex : A1, nm1 = s ? A1 : A0;
    const BondT jm0 = s ? B0 : Jex, jm1 = s ? B1 : B0;

    const SweepRng g = make_sweep_rng(a.seed, sweep_time(a), (uint32_t)a.colour);
    const uint32_t site0 = (4 * k + s) + L * (y + L * z);
    const uint4 r = sweep_random4(g, site0); // the thread's two words are one pair (xh = 2k, 2k + 1): one block
    ulonglong2 out;
    out.x = metropolis_word<BondT, ALWAYS, false, HB>(sg0, np0, nm0, yp0, ym0, zp0, zm0, jx0, jm0, jy0, by0, jz0, bz0, r.x, r.y, a.th);
    out.y = metropolis_word<BondT, ALWAYS, false, HB>(sg1, np1, nm1, yp1, ym1, zp1, zm1, jx1, jm1, jy1, by1, jz1, bz1, r.z, r.w, a.th);
    *(ulonglong2 *)(a.own + i0) = out;
}

__global__ void k_bump_time(uint64_t *d_time, uint32_t n) { *d_time += n; }

// ---------------------------------------------------------------------------------------------
// ROWS: a warp owns whole x-rows (L/4 lanes per row, two words per lane) and marches M rows along y, keeping
// the other colour's rows y-1, y, y+1 in registers (each is loaded once instead of three times).  The row
// phase s = (colour ^ (y + z)) & 1 alternates along y, so the march is unrolled by two with s a compile-time
// constant: no selects, and the one x-neighbour word outside the lane's aligned pair comes from the adjacent
// lane by a warp shuffle (the periodic wrap in x is a rotation inside the row's lane group).
// L in {16, 32, 64, 128} (L/4 lanes per row must divide the warp), L a compile-time constant so every row
// stride is an immediate.  A warp with several rows (L < 128) takes rows of equal z parity, which keeps s
// warp-uniform.
// ---------------------------------------------------------------------------------------------

// spins of the other colour: read-only path (one launch per colour), or L2-coherent loads when other CTAs rewrite
// them inside the same launch (ROWS_PERSISTENT)
template <bool COHERENT> __device__ __forceinline__ ulonglong2 ld_oth(const uint64_t *p)
{
    return COHERENT ? __ldcg((const ulonglong2 *)p) : __ldg((const ulonglong2 *)p);
}

template <int L, int M, int S0, typename BondT, bool ALWAYS, bool HB, bool COHERENT = false>
__device__ __forceinline__ void march_rows(const SweepArgs &a, const SweepRng &g, const unsigned y0, const unsigned z,
                                           const unsigned k, const int lane_m, const int lane_p)
{
    constexpr unsigned Lh = L / 2, Nh = (unsigned)L * L * L / 2, ZS = Lh * L; // row and plane strides (words)
    const BondT *__restrict__ Jc = (const BondT *)a.Jc;
    const BondT *__restrict__ Jo = (const BondT *)a.Jo;
    const unsigned zb = ZS * z + 2 * k, zbm = ZS * ((z - 1) & (L - 1)) + 2 * k, zbp = ZS * ((z + 1) & (L - 1)) + 2 * k;
    ulonglong2 Pm = ld_oth<COHERENT>(a.oth + zb + Lh * ((y0 - 1) & (L - 1)));
    ulonglong2 P0 = ld_oth<COHERENT>(a.oth + zb + Lh * y0);
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const unsigned y = y0 + m, row = zb + Lh * y;
        const ulonglong2 own = *(const ulonglong2 *)(a.own + row);
        const ulonglong2 Pp = ld_oth<COHERENT>(a.oth + zb + Lh * ((y + 1) & (L - 1)));
        const ulonglong2 Zm = ld_oth<COHERENT>(a.oth + zbm + Lh * y);
        const ulonglong2 Zp = ld_oth<COHERENT>(a.oth + zbp + Lh * y);
        const typename Pair<BondT>::type jx = ldg_pair<BondT>(Jc + row), jy = ldg_pair<BondT>(Jc + Nh + row),
                                         jz = ldg_pair<BondT>(Jc + 2 * Nh + row), bx = ldg_pair<BondT>(Jo + row),
                                         by = ldg_pair<BondT>(Jo + Nh + zb + Lh * ((y - 1) & (L - 1))),
                                         bz = ldg_pair<BondT>(Jo + 2 * Nh + zbm + Lh * y);
        const uint32_t site0 = 4 * k + L * (y + L * z);
        ulonglong2 out;
        if (((m & 1) ^ S0) == 0)
            out = update_pair<0, BondT, ALWAYS, false, HB>(own, P0, Pm, Pp, Zm, Zp, jx, jy, jz, bx, by, bz, site0, g, a.th, lane_m, lane_p);
        else
            out = update_pair<1, BondT, ALWAYS, false, HB>(own, P0, Pm, Pp, Zm, Zp, jx, jy, jz, bx, by, bz, site0 + 1, g, a.th, lane_m, lane_p);
        *(ulonglong2 *)(a.own + row) = out;
        Pm = P0;
        P0 = Pp;
    }
}

template <int L, int M, typename BondT, bool ALWAYS, bool HB>
__global__ void __launch_bounds__(128) k_sweep_rows(const SweepArgs a)
{
    pdl_launch_dependents();
    constexpr unsigned RL = L / 4, G = 32 / RL; // lanes per row, rows per warp
    constexpr unsigned YC = L / M;              // y-chunks
    const unsigned lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned k = lane % RL, grp = lane / RL;
    const unsigned zg = warp / YC, yc = warp - zg * YC; // consecutive warps: the y-chunks of one z group
    if (zg >= L / G) return;
    const unsigned zpar = zg & 1, z = 2 * (G * (zg >> 1) + grp) + zpar, y0 = yc * M;
    const int lane_m = (int)((lane & ~(RL - 1)) | ((k - 1) & (RL - 1))), lane_p = (int)((lane & ~(RL - 1)) | ((k + 1) & (RL - 1)));
    pdl_wait(); // the previous half-sweep is complete; spins of the other colour through L2 (the read-only path may predate it)
    const SweepRng g = make_sweep_rng(a.seed, sweep_time(a), (uint32_t)a.colour);
    if (((a.colour ^ zpar ^ y0) & 1u) == 0) // phase of row y0: warp-uniform
        march_rows<L, M, 0, BondT, ALWAYS, HB, true>(a, g, y0, z, k, lane_m, lane_p);
    else
        march_rows<L, M, 1, BondT, ALWAYS, HB, true>(a, g, y0, z, k, lane_m, lane_p);
}

// ROWS_PERSISTENT (L = 16, 32, 64; SURVEY 8(f) NEXT-2 "grid-barrier persistent kernels for L <= 64"): all 2n
// half-sweeps of one ea_sweep(n) call in ONE cooperative launch; the colour barrier is a grid-wide barrier
// (~1.2 us) instead of a kernel boundary (~2-2.8 us per graph node at these sizes, which are launch-bound).
// Same geometry as k_sweep_rows, so a row is always updated by the same thread; the other colour's rows are
// rewritten by other CTAs between steps and are therefore read with L2-coherent loads.
// MEASURED (B200): 1.93 / 4.05 / 4.29 us per half-sweep at L = 16 / 32 / 64 against 2.05 / 2.53 / 2.79 us for the
// CUDA-graph replays of k_sweep_rows: the grid barrier over 32-256 CTAs costs more than the graph node it replaces.
// Kept as an explicit option (bit-identical, tested); AUTO does not choose it.
template <int L, int M, typename BondT, bool ALWAYS>
__global__ void __launch_bounds__(128) k_sweep_rows_persistent(SweepArgs a, uint64_t *spins, const BondT *bonds, const uint32_t n_half)
{
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    constexpr unsigned RL = L / 4, G = 32 / RL, YC = L / M, Nh = (unsigned)L * L * L / 2;
    const unsigned lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned k = lane % RL, grp = lane / RL;
    const unsigned zg = warp / YC, yc = warp - zg * YC;
    const bool active = zg < L / G;
    const unsigned zpar = zg & 1, z = 2 * (G * (zg >> 1) + grp) + zpar, y0 = yc * M;
    const int lane_m = (int)((lane & ~(RL - 1)) | ((k - 1) & (RL - 1))), lane_p = (int)((lane & ~(RL - 1)) | ((k + 1) & (RL - 1)));
    const uint64_t t0 = a.t;
    for (uint32_t h = 0; h < n_half; ++h) {
        const int c = h & 1;
        a.colour = c;
        a.own = spins + (size_t)c * Nh;
        a.oth = spins + (size_t)(1 - c) * Nh;
        a.Jc = bonds + (size_t)c * 3 * Nh;
        a.Jo = bonds + (size_t)(1 - c) * 3 * Nh;
        if (active) {
            const SweepRng g = make_sweep_rng(a.seed, t0 + (h >> 1), (uint32_t)c);
            if ((c ^ zpar) == 0) march_rows<L, M, 0, BondT, ALWAYS, false, true>(a, g, y0, z, k, lane_m, lane_p);
            else march_rows<L, M, 1, BondT, ALWAYS, false, true>(a, g, y0, z, k, lane_m, lane_p);
        }
        grid.sync(); // colour barrier, with the memory fence that publishes this step's rows
    }
}

template <int L, typename BondT, bool ALWAYS>
static cudaError_t launch_rows_persistent_L(ea_sim *s, SweepArgs &a, uint32_t n, cudaStream_t st)
{
    constexpr int M = (L >= 128) ? 4 : 2, G = 32 / (L / 4);
    constexpr unsigned warps = (L / M) * (L / G), block = 128, grid = (warps * 32 + block - 1) / block;
    auto kern = k_sweep_rows_persistent<L, M, BondT, ALWAYS>;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, block, 0);
    if (e != cudaSuccess) return e;
    if ((unsigned)per_sm * (unsigned)s->n_sm < grid) return cudaErrorCooperativeLaunchTooLarge;
    uint64_t *spins = s->spins;
    const BondT *bonds = (const BondT *)s->bonds;
    uint32_t n_half = 2 * n;
    void *args[] = {&a, &spins, &bonds, &n_half};
    return cudaLaunchCooperativeKernel((void *)kern, dim3(grid), dim3(block), args, 0, st);
}

template <typename BondT>
static cudaError_t launch_rows_persistent_typed(ea_sim *s, SweepArgs &a, uint32_t n, cudaStream_t st)
{
    const bool always = a.th.always[0] | a.th.always[1] | a.th.always[2];
    switch (s->lat.L) {
    case 16: return always ? launch_rows_persistent_L<16, BondT, true>(s, a, n, st) : launch_rows_persistent_L<16, BondT, false>(s, a, n, st);
    case 32: return always ? launch_rows_persistent_L<32, BondT, true>(s, a, n, st) : launch_rows_persistent_L<32, BondT, false>(s, a, n, st);
    case 64: return always ? launch_rows_persistent_L<64, BondT, true>(s, a, n, st) : launch_rows_persistent_L<64, BondT, false>(s, a, n, st);
    default: return cudaErrorInvalidValue;
    }
}

bool rows_persistent_valid(int L) { return L == 16 || L == 32 || L == 64; }

// n sweeps (Metropolis) from sweep index t0 in one cooperative launch
cudaError_t launch_sweeps_rows_persistent(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st)
{
    SweepArgs a;
    a.lat = s->lat;
    a.colour = 0;
    a.own = nullptr; a.oth = nullptr; a.Jc = nullptr; a.Jo = nullptr; // set per step on the device
    a.seed = s->seed;
    a.t = t0;
    a.d_time = nullptr;
    a.t_offset = 0;
    a.th = s->th;
    cudaError_t e = s->n_replicas == 2 ? launch_rows_persistent_typed<uint32_t>(s, a, n, st)
                                       : launch_rows_persistent_typed<uint64_t>(s, a, n, st);
    if (e == cudaSuccess) s->count_launch();
    return e;
}

// rows a warp marches along y: 4 at L = 128 (the register window pays), 2 below (measured with one row per warp: L = 64 2.82
// against 2.47 us per half-sweep, L = 16 1.57 against 2.00 -- but L <= 32 runs the SMALL kernel anyway)
template <int L> struct ROWS_M { static constexpr int value = L >= 128 ? 4 : 2; };

template <int L, typename BondT, bool ALWAYS, bool HB>
static void launch_rows(const SweepArgs &a, cudaStream_t st)
{
    constexpr int M = ROWS_M<L>::value, G = 32 / (L / 4);
    constexpr unsigned warps = (L / M) * (L / G), block = 128, grid = (warps * 32 + block - 1) / block;
    launch_pdl(k_sweep_rows<L, M, BondT, ALWAYS, HB>, dim3(grid), dim3(block), st, a);
}

// ---------------------------------------------------------------------------------------------
template <typename BondT, bool ALWAYS, bool HB>
static cudaError_t launch_typed(ea_sim *s, const SweepArgs &a, cudaStream_t st)
{
    const Lattice &lat = s->lat;
    const bool pow2 = lat.log2L >= 0;
    // RESIDENT / SMALL: single half-sweeps and short calls go as per-colour launches of the best variant valid for L
    const bool rows_ok = lat.L == 16 || lat.L == 32 || lat.L == 64 || lat.L == 128;
    const int kernel = s->kernel == EA_KERNEL_SMALL ? (rows_ok ? (int)EA_KERNEL_ROWS : (int)EA_KERNEL_VEC2) : s->kernel;
    if (kernel == EA_KERNEL_ROWS || kernel == EA_KERNEL_RESIDENT || kernel == EA_KERNEL_ROWS_PERSISTENT) {
        switch (lat.L) {
        case 16: launch_rows<16, BondT, ALWAYS, HB>(a, st); break;
        case 32: launch_rows<32, BondT, ALWAYS, HB>(a, st); break;
        case 64: launch_rows<64, BondT, ALWAYS, HB>(a, st); break;
        case 128: launch_rows<128, BondT, ALWAYS, HB>(a, st); break;
        default: return cudaErrorInvalidValue;
        }
    } else if (kernel == EA_KERNEL_VEC2) {
        unsigned n = lat.Nh / 2, block = 256, grid = (n + block - 1) / block;
        if (pow2) launch_pdl(k_sweep_vec2<BondT, true, ALWAYS, HB>, dim3(grid), dim3(block), st, a);
        else launch_pdl(k_sweep_vec2<BondT, false, ALWAYS, HB>, dim3(grid), dim3(block), st, a);
    } else {
        unsigned n = lat.Nh, block = 256, grid = (n + block - 1) / block;
        if (pow2) launch_pdl(k_sweep_scalar<BondT, true, ALWAYS, HB>, dim3(grid), dim3(block), st, a);
        else launch_pdl(k_sweep_scalar<BondT, false, ALWAYS, HB>, dim3(grid), dim3(block), st, a);
    }
    s->count_launch();
    return cudaGetLastError();
}

template <typename BondT>
static cudaError_t launch_typed(ea_sim *s, const SweepArgs &a, cudaStream_t st)
{
    if (s->dynamics == EA_DYN_HEATBATH) return launch_typed<BondT, false, true>(s, a, st); // carries its own always-masks
    const bool always = a.th.always[0] | a.th.always[1] | a.th.always[2]; // T = inf: some thr == 2^32
    return always ? launch_typed<BondT, true, false>(s, a, st) : launch_typed<BondT, false, false>(s, a, st);
}

cudaError_t launch_half_sweep(ea_sim *s, int parity, uint64_t t, const uint64_t *d_time, uint32_t t_offset,
                              cudaStream_t st)
{
    if (s->n_samples < EA_LANES) return launch_half_sweep_fold(s, parity, t, d_time, t_offset, st); // M < 64 (ea_fold.cu)
    SweepArgs a;
    a.lat = s->lat;
    a.colour = parity;
    a.own = s->spins_c(parity);
    a.oth = s->spins_c(1 - parity);
    const size_t plane = (size_t)3 * s->lat.Nh * s->bond_bytes();
    a.Jc = (const char *)s->bonds + (size_t)parity * plane;
    a.Jo = (const char *)s->bonds + (size_t)(1 - parity) * plane;
    a.seed = s->seed;
    a.t = t;
    a.d_time = d_time;
    a.t_offset = t_offset;
    a.th = s->th;
    return s->n_replicas == 2 ? launch_typed<uint32_t>(s, a, st) : launch_typed<uint64_t>(s, a, st);
}

// ---------------------------------------------------------------------------------------------
// BATCH ("batched multi-sim driver"): K independent small sims (same L, same bond width, same
// dynamics; own p, T, seed, t) in ONE launch per colour -- blockIdx.y picks the sim.  Lattices of L <= 64 are
// launch-bound (a 32^3 half-sweep is a 32-CTA kernel behind a 2 us launch), and concurrent streams hit the launch
// rate of the device (~0.4 us per kernel); fusing K sims into one grid removes both limits.
// ---------------------------------------------------------------------------------------------
template <int L, int M, typename BondT, bool ALWAYS, bool HB>
__global__ void __launch_bounds__(128) k_sweep_rows_batch(const SweepArgs *__restrict__ args, const uint32_t t_offset)
{
    SweepArgs a = args[blockIdx.y];
    a.t_offset = t_offset;
    constexpr unsigned RL = L / 4, G = 32 / RL, YC = L / M;
    const unsigned lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned k = lane % RL, grp = lane / RL;
    const unsigned zg = warp / YC, yc = warp - zg * YC;
    if (zg >= L / G) return;
    const unsigned zpar = zg & 1, z = 2 * (G * (zg >> 1) + grp) + zpar, y0 = yc * M;
    const int lane_m = (int)((lane & ~(RL - 1)) | ((k - 1) & (RL - 1))), lane_p = (int)((lane & ~(RL - 1)) | ((k + 1) & (RL - 1)));
    const SweepRng g = make_sweep_rng(a.seed, sweep_time(a), (uint32_t)a.colour);
    if ((a.colour ^ zpar) == 0) march_rows<L, M, 0, BondT, ALWAYS, HB>(a, g, y0, z, k, lane_m, lane_p);
    else march_rows<L, M, 1, BondT, ALWAYS, HB>(a, g, y0, z, k, lane_m, lane_p);
}

__global__ void k_bump_time_batch(uint64_t *const *d_times, unsigned n_sims, uint32_t n)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_sims) *d_times[i] += n;
}

template <int L, typename BondT, bool ALWAYS, bool HB>
static void launch_rows_batch_L(const SweepArgs *d_args, unsigned n_sims, uint32_t t_offset, cudaStream_t st)
{
    constexpr int M = 2, G = 32 / (L / 4);
    constexpr unsigned warps = (L / M) * (L / G), block = 128, grid = (warps * 32 + block - 1) / block;
    k_sweep_rows_batch<L, M, BondT, ALWAYS, HB><<<dim3(grid, n_sims), block, 0, st>>>(d_args, t_offset);
}

template <typename BondT, bool ALWAYS, bool HB>
static cudaError_t launch_rows_batch_typed(int L, const SweepArgs *d_args, unsigned n_sims, uint32_t t_offset, cudaStream_t st)
{
    switch (L) {
    case 16: launch_rows_batch_L<16, BondT, ALWAYS, HB>(d_args, n_sims, t_offset, st); break;
    case 32: launch_rows_batch_L<32, BondT, ALWAYS, HB>(d_args, n_sims, t_offset, st); break;
    case 64: launch_rows_batch_L<64, BondT, ALWAYS, HB>(d_args, n_sims, t_offset, st); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// host copy of the launch arguments of one sim for one colour (time from the sim's device clock + t_offset)
void fill_batch_args(const ea_sim *s, int parity, void *out /* SweepArgs */)
{
    SweepArgs a;
    a.lat = s->lat;
    a.colour = parity;
    a.own = s->spins_c(parity);
    a.oth = s->spins_c(1 - parity);
    const size_t plane = (size_t)3 * s->lat.Nh * s->bond_bytes();
    a.Jc = (const char *)s->bonds + (size_t)parity * plane;
    a.Jo = (const char *)s->bonds + (size_t)(1 - parity) * plane;
    a.seed = s->seed;
    a.t = 0;
    a.d_time = s->d_time;
    a.t_offset = 0;
    a.th = s->th;
    memcpy(out, &a, sizeof(a));
}
size_t batch_args_bytes() { return sizeof(SweepArgs); }

cudaError_t launch_half_sweep_batch(int L, int n_replicas, bool always, bool heatbath, const void *d_args, unsigned n_sims,
                                    uint32_t t_offset, cudaStream_t st)
{
    const SweepArgs *a = (const SweepArgs *)d_args;
    if (n_replicas == 2) {
        if (heatbath) return launch_rows_batch_typed<uint32_t, false, true>(L, a, n_sims, t_offset, st);
        return always ? launch_rows_batch_typed<uint32_t, true, false>(L, a, n_sims, t_offset, st)
                      : launch_rows_batch_typed<uint32_t, false, false>(L, a, n_sims, t_offset, st);
    }
    if (heatbath) return launch_rows_batch_typed<uint64_t, false, true>(L, a, n_sims, t_offset, st);
    return always ? launch_rows_batch_typed<uint64_t, true, false>(L, a, n_sims, t_offset, st)
                  : launch_rows_batch_typed<uint64_t, false, false>(L, a, n_sims, t_offset, st);
}

cudaError_t launch_bump_time_batch(uint64_t *const *d_times, unsigned n_sims, uint32_t n, cudaStream_t st)
{
    k_bump_time_batch<<<(n_sims + 127) / 128, 128, 0, st>>>(d_times, n_sims, n);
    return cudaGetLastError();
}

cudaError_t launch_bump_time(ea_sim *s, uint32_t n, cudaStream_t st)
{
    k_bump_time<<<1, 1, 0, st>>>(s->d_time, n);
    s->count_launch();
    return cudaGetLastError();
}

} // namespace ea

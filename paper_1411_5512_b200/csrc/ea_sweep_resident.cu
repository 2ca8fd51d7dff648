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
#include <utility>
#include <vector>

#include "ea_internal.h"
#include "ea_sweep_common.cuh"

namespace ea {

struct ResidentArgs {
    uint64_t *spins;     // [2][Nh]
    const void *bonds;   // BondT [2][3][Nh]
    uint32_t k0[10], k1[10]; // Philox round keys of the seed (C-A6)
    uint64_t t0;         // first sweep index
    uint32_t n_half;     // half-steps to run (2 per sweep)
    uint32_t epoch0;     // flag value before this launch; step h publishes epoch0 + h + 1
    unsigned *flags;     // [G][32]: one 128-byte line per CTA
    unsigned *abort_flag;// set by any CTA whose wait timed out; everybody then leaves
    unsigned long long timeout_ns; // a neighbour that never shows up: give up after this long
    Thresholds th;
};

template <int L_, int TY_, int TZ_, int CW_, int UNROLL_> struct ResidentGeom {
    static constexpr int L = L_, TY = TY_, TZ = TZ_;
    static constexpr int Lh = L / 2;                 // words per colour row
    static constexpr int NTY = L / TY, NTZ = L / TZ; // tiles along y, z
    static constexpr int G = NTY * NTZ;              // CTAs
    static constexpr int ROWS = TY * TZ;             // rows updated per CTA per half-step
    static constexpr int HY = TY + 2, HZ = TZ + 2;   // with halo ring
    static constexpr int CW = CW_;                   // compute warps
    static constexpr int UNROLL = UNROLL_;           // row pairs unrolled per loop iteration of a half-step (code size vs. scheduling freedom)
    static constexpr int THREADS = (CW + 1) * 32;    // + one producer warp
    static constexpr int NB = ROWS - (TY - 2) * (TZ - 2); // boundary rows
    static constexpr unsigned HALO_BYTES = (2 * TY + 2 * TZ) * Lh * 8;
    static constexpr size_t SPIN_BYTES = (size_t)2 * HZ * HY * Lh * 8;
    static constexpr size_t SMEM_BYTES = SPIN_BYTES + 16 /*mbarrier*/ + ROWS * 16 /*row descriptors*/;
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
constexpr uint32_t RARE_THR2_MAX = 0x04000000u; // P(r < thr[2]) < 1/64: the warp-level branch of metropolis_word pays

// Row schedule of one CTA (built on the host, build_row_table): compute warp w updates rows row[w][0..RPW-1]
// (yy | zz << 8, tile coordinates 1..TY, 1..TZ), boundary rows first (n_bnd[w] of them), and consecutive rows
// of a warp alternate in (yy + zz) parity starting from phi[w] -- so the row phase s = (colour ^ y ^ z) & 1 of
// every row is a compile-time constant once the warp-uniform (colour ^ phi[w]) is known.
template <typename G> struct RowTable {
    uint16_t row[G::CW][G::ROWS / G::CW];
    uint8_t n_bnd[G::CW];
    uint8_t phi[G::CW];
};

template <typename BondT> struct RowBonds { typename Pair<BondT>::type jx, jy, jz, bx, by, bz; };

// Row descriptor (shared memory, one per (compute warp, row slot), written once in the prologue):
//   x = byte offset of row (zz, yy) inside a colour plane of the tile
//   y = word offset of row (y, z) inside a colour plane of the global arrays, Lh * (y + L * z)
//   z = Nh + offset of row (y-1, z),  w = 2 Nh + offset of row (y, z-1)    (periodic) -- the backward y / z bonds
template <typename G>
__device__ __forceinline__ uint4 make_row_desc(unsigned yy, unsigned zz, unsigned y0, unsigned z0)
{
    constexpr unsigned Lh = G::Lh, L = G::L, Nh = (unsigned)L * L * L / 2;
    const unsigned y = y0 + yy - 1, z = z0 + zz - 1;
    uint4 d;
    d.x = (zz * G::HY + yy) * Lh * 8;
    d.y = Lh * (y + L * z);
    d.z = Nh + Lh * (((y - 1) & (L - 1)) + L * z);
    d.w = 2 * Nh + Lh * (y + L * ((z - 1) & (L - 1)));
    return d;
}

// Row addresses are "64-bit per-lane base + 32-bit element offset from the row descriptor": one IMAD.WIDE.U32 on the
// fma pipe (the kernel is bound by the alu pipe, where a 64-bit add would cost an IADD3 / IADD3.X pair per row).
// The base is a full 64-bit pointer, so the arrays may lie anywhere in the address space.
struct Ptr32 {
    const char *base;
    __device__ __forceinline__ Ptr32() {}
    __device__ __forceinline__ explicit Ptr32(const void *p) : base((const char *)p) {}
    template <typename T> __device__ __forceinline__ T *at(unsigned elem_off) const
    {
        return (T *)(base + (size_t)elem_off * sizeof(T));
    }
};

// Jc_l / Jo_l: bond planes of the updated / the other colour, already offset by the lane's 2k words
template <typename BondT>
__device__ __forceinline__ RowBonds<BondT> load_row_bonds(const Ptr32 Jc_l, const Ptr32 Jo_l, const uint4 d,
                                                          const unsigned Nh)
{
    RowBonds<BondT> b;
    const BondT *pc = Jc_l.at<const BondT>(d.y);
    b.jx = ldg_pair<BondT>(pc);
    b.jy = ldg_pair<BondT>(pc + Nh);
    b.jz = ldg_pair<BondT>(pc + 2 * Nh);
    b.bx = ldg_pair<BondT>(Jo_l.at<const BondT>(d.y));
    b.by = ldg_pair<BondT>(Jo_l.at<const BondT>(d.z));
    b.bz = ldg_pair<BondT>(Jo_l.at<const BondT>(d.w));
    return b;
}

// per-step, per-lane context of a compute warp
struct ResidentStep {
    const unsigned char *s_oth; // tile plane of colour 1-c + 16 * lane
    unsigned char *s_own;       // tile plane of colour c + 16 * lane
    Ptr32 g_own;                // global plane of colour c + 2 * lane
    unsigned k;
    int lane_m, lane_p;
};

// the four random numbers of the lane's two words of a row (d.y = row offset, S = row phase; C-A7): independent of the
// spins, so they are drawn one row ahead and their IMAD.WIDE chain (fma pipe) overlaps the LOP3 logic (alu pipe)
// of the row before
__device__ __forceinline__ uint4 row_random(const SweepRng &g, const unsigned k, const unsigned S, const uint4 d)
{
    // canonical site = x + L (y + L z), L = 2 Lh; the lane's two words (xh = 2k, 2k + 1) are one pair: one block
    return sweep_random4(g, 4 * k + S + 2 * d.y);
}

// one row of colour c with compile-time phase S; publishes it to global when `publish`
template <int S, typename G, typename BondT, bool ALWAYS, bool RARE, bool HB>
__device__ __forceinline__ void resident_row(const ResidentStep &x, const uint4 d, const RowBonds<BondT> &bd,
                                             const uint4 r, const Thresholds &th, const bool publish)
{
    constexpr int ROWB = G::Lh * 8, PLANEB = G::HY * G::Lh * 8; // smem strides: next y row, next z plane
    unsigned char *own_row = x.s_own + d.x;
    const unsigned char *o = x.s_oth + d.x;
    const ulonglong2 own = *(const ulonglong2 *)own_row;
    const ulonglong2 P0 = *(const ulonglong2 *)o;
    const ulonglong2 Pm = *(const ulonglong2 *)(o - ROWB);
    const ulonglong2 Pp = *(const ulonglong2 *)(o + ROWB);
    const ulonglong2 Zm = *(const ulonglong2 *)(o - PLANEB);
    const ulonglong2 Zp = *(const ulonglong2 *)(o + PLANEB);
    const ulonglong2 out = update_pair_r<S, BondT, ALWAYS, RARE, HB>(own, P0, Pm, Pp, Zm, Zp, bd.jx, bd.jy, bd.jz, bd.bx, bd.by,
                                                                 bd.bz, r, th, x.lane_m, x.lane_p);
    *(ulonglong2 *)own_row = out;
    if (publish) *x.g_own.at<ulonglong2>(d.y / 2) = out;
}

// all rows of one compute warp for one half-step; S0 = phase of the warp's first row.  Carried across rows and
// steps: nxt = bond words of the next row, rnx = random numbers of the next row (gn = stream of the next step).
template <int S0, typename G, typename BondT, bool ALWAYS, bool RARE, bool HB>
__device__ __forceinline__ void resident_step(const ResidentStep &x, const uint4 *__restrict__ desc, const int n_bnd,
                                              RowBonds<BondT> &nxt, uint4 &rnx, const Ptr32 Jc_l, const Ptr32 Jo_l,
                                              const SweepRng &g, const SweepRng &gn, const Thresholds &th)
{
    constexpr int RPW = G::ROWS / G::CW;
    constexpr unsigned Nh = (unsigned)G::L * G::L * G::L / 2;
    static_assert(RPW % 2 == 0, "rows are taken two at a time (phases S0, 1 - S0)");
    // a warp has at most NB_HI boundary rows (the slowest warps of the boundary phase have exactly NB_HI, and the
    // producer waits for all of them): ONE arrive after row NB_HI - 1, and only the first NB_HI rows carry the publish
    // store.  (An asm statement is a scheduling fence: every other row is free to interleave with its neighbours.)
    constexpr int NB_HI = (G::NB + G::CW - 1) / G::CW;
    static_assert(NB_HI >= 1 && NB_HI <= RPW, "the arrive must sit inside the row loop");
#pragma unroll(G::UNROLL)
    for (int i = 0; i < RPW; i += 2) {
        const bool last = i + 2 >= RPW;
        const uint4 d0 = desc[i], d1 = desc[i + 1], d2 = desc[last ? 0 : i + 2];
        const RowBonds<BondT> b0 = nxt;
        const uint4 r0 = rnx;
        const RowBonds<BondT> b1 = load_row_bonds<BondT>(Jc_l, Jo_l, d1, Nh);
        const uint4 r1 = row_random(g, x.k, 1 - S0, d1);
        resident_row<S0, G, BondT, ALWAYS, RARE, HB>(x, d0, b0, r0, th, (G::UNROLL * 2 < RPW || i < NB_HI) && i < n_bnd);
        if (i + 1 == NB_HI) named_bar_arrive(BAR_BOUNDARY, G::THREADS); // every warp's boundary rows are done by now
        // the row after next; for the last pair that is the first row of the next half-step: the colours swap
        // roles, the stream moves on, and the phase of row 0 flips with the colour
        if (!last) {
            nxt = load_row_bonds<BondT>(Jc_l, Jo_l, d2, Nh);
            rnx = row_random(g, x.k, S0, d2);
        } else {
            nxt = load_row_bonds<BondT>(Jo_l, Jc_l, d2, Nh);
            rnx = row_random(gn, x.k, 1 - S0, d2);
        }
        resident_row<1 - S0, G, BondT, ALWAYS, RARE, HB>(x, d1, b1, r1, th, (G::UNROLL * 2 < RPW || i + 1 < NB_HI) && i + 1 < n_bnd);
        if (i + 2 == NB_HI) named_bar_arrive(BAR_BOUNDARY, G::THREADS);
    }
}

template <typename G, typename BondT, bool ALWAYS, bool RARE, bool HB>
__global__ void __launch_bounds__(G::THREADS, 1) k_sweep_resident(const ResidentArgs a, const RowTable<G> tab)
{
    constexpr int L = G::L, Lh = G::Lh, TY = G::TY, TZ = G::TZ, HY = G::HY, HZ = G::HZ, CW = G::CW, ROWS = G::ROWS;
    constexpr unsigned Nh = (unsigned)L * L * L / 2;
    constexpr int RPW = ROWS / CW; // rows per compute warp per half-step
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *tile = (uint64_t *)smem_raw;                       // [2][HZ][HY][Lh]
    uint64_t *halo_bar = (uint64_t *)(smem_raw + G::SPIN_BYTES); // mbarrier: halo of the next step has landed
    uint4 *rowdesc = (uint4 *)(smem_raw + G::SPIN_BYTES + 16);   // [CW][RPW] row descriptors

    const unsigned tid = threadIdx.x, lane = tid & 31;
    const unsigned warp = __shfl_sync(0xffffffffu, tid >> 5, 0); // provably warp-uniform: no divergence guards around the shuffles
    const unsigned b = blockIdx.x, ty = b % G::NTY, tz = b / G::NTY;
    const unsigned y0 = ty * TY, z0 = tz * TZ;
    auto tile_at = [&](int c, int zz, int yy) -> uint64_t * { return tile + ((size_t)(c * HZ + zz) * HY + yy) * Lh; };

    // ---- prologue: barrier, tile + halo ring of both colours from global -------------------------------
    if (tid < (unsigned)ROWS)
        rowdesc[tid] = make_row_desc<G>(tab.row[tid / RPW][tid % RPW] & 0xff, tab.row[tid / RPW][tid % RPW] >> 8, y0, z0);
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
        // the halo copy of this lane (2 z-faces of TY rows, then 2 y-face rows per tile plane): offsets within a colour
        const unsigned zlo = (z0 - 1) & (L - 1), zhi = (z0 + TZ) & (L - 1);
        const unsigned ylo = (y0 - 1) & (L - 1), yhi = (y0 + TY) & (L - 1);
        unsigned cp_src = 0, cp_dst = 0, cp_bytes = 0; // word offsets
        if (lane < 2) {
            cp_src = Lh * (y0 + L * (lane ? zhi : zlo));
            cp_dst = ((lane ? HZ - 1 : 0) * HY + 1) * Lh;
            cp_bytes = TY * Lh * 8;
        } else if (lane < 2 + 2 * TZ) {
            const unsigned j = lane - 2, zz = 1 + (j >> 1), hi = j & 1;
            cp_src = Lh * ((hi ? yhi : ylo) + L * (z0 + zz - 1));
            cp_dst = (zz * HY + (hi ? HY - 1 : 0)) * Lh;
            cp_bytes = Lh * 8;
        }
        static_assert(2 + 2 * TZ <= 32, "one halo copy per producer lane");
        for (uint32_t h = 0; h < a.n_half; ++h) {
            const int c = h & 1;
            named_bar_sync(BAR_BOUNDARY, G::THREADS); // boundary rows of step h are in smem and in global
            const unsigned epoch = a.epoch0 + h + 1;
            if (lane == 0) st_release_gpu(a.flags + b * 32, epoch); // release: cumulative over the CTA's stores
            if (h + 1 == a.n_half) break;
            bool ok = true;
            if (lane < 4) {
                const unsigned *f = a.flags + nb_tile * 32;
                const unsigned long long t_start = globaltimer_ns();
                unsigned spins = 0;
                while ((int)(ld_acquire_gpu(f) - epoch) < 0) {
                    if ((++spins & 63u) == 0) {
                        if (*(volatile unsigned *)a.abort_flag || globaltimer_ns() - t_start > a.timeout_ns) {
                            ok = false;
                            break;
                        }
                    }
                }
            }
            ok = __all_sync(0xffffffffu, ok);
            // on a time-out: raise the abort flag (every CTA stops waiting), keep going with stale halos so that
            // all barriers still complete; the host finds the flag at its next synchronisation and reports it
            if (!ok && lane == 0) atomicExch(a.abort_flag, 1u);
            if (lane == 0) mbar_arrive_expect_tx(halo_bar, G::HALO_BYTES);
            __syncwarp();
            if (cp_bytes) {
                asm volatile("fence.proxy.async;" ::: "memory");
                bulk_g2s(tile + (size_t)c * HZ * HY * Lh + cp_dst, a.spins + (size_t)c * Nh + cp_src, cp_bytes, halo_bar);
            }
        }
    } else {
        // ---- compute warps -----------------------------------------------------------------------------
        const int n_bnd = tab.n_bnd[warp];
        const unsigned phi = tab.phi[warp];
        const uint4 *__restrict__ desc = rowdesc + warp * RPW;
        ResidentStep x;
        x.k = lane;
        x.lane_m = (int)((lane - 1) & 31);
        x.lane_p = (int)((lane + 1) & 31);
        SweepRng g;
#pragma unroll
        for (int r = 0; r < 10; ++r) { g.k0[r] = a.k0[r]; g.k1[r] = a.k1[r]; }

        // software pipeline: the bond words of the next row are always in flight
        RowBonds<BondT> nxt = load_row_bonds<BondT>(Ptr32(bonds + 2 * lane), Ptr32(bonds + (size_t)3 * Nh + 2 * lane), desc[0], Nh);
        sweep_rng_set_time(g, a.t0, 0u);
        uint4 rnx = row_random(g, lane, phi & 1u, desc[0]); // phase of row 0 in step 0 (colour 0) is phi
        for (uint32_t h = 0; h < a.n_half; ++h) {
            const int c = h & 1;
            sweep_rng_set_time(g, a.t0 + (h >> 1), (uint32_t)c);
            SweepRng gn = g;
            sweep_rng_set_time(gn, a.t0 + ((h + 1) >> 1), (uint32_t)(1 - c));
            const Ptr32 Jc_l(bonds + (size_t)c * 3 * Nh + 2 * lane), Jo_l(bonds + (size_t)(1 - c) * 3 * Nh + 2 * lane);
            x.s_own = (unsigned char *)(tile + (size_t)c * HZ * HY * Lh) + 16 * lane;
            x.s_oth = (const unsigned char *)(tile + (size_t)(1 - c) * HZ * HY * Lh) + 16 * lane;
            x.g_own = Ptr32(a.spins + (size_t)c * Nh + 2 * lane);
            if (h > 0) { // halo of colour 1-c, pulled in during step h-1
                const unsigned parity = (h - 1) & 1;
                while (!mbar_try_wait(halo_bar, parity)) { } // always completes: the producer arms it even on abort
            }
            // y0, z0 are even, so the phase of row i is (c ^ phi ^ i) & 1
            if (((unsigned)c ^ phi) & 1u) resident_step<1, G, BondT, ALWAYS, RARE, HB>(x, desc, n_bnd, nxt, rnx, Jc_l, Jo_l, g, gn, a.th);
            else resident_step<0, G, BondT, ALWAYS, RARE, HB>(x, desc, n_bnd, nxt, rnx, Jc_l, Jo_l, g, gn, a.th);
            named_bar_sync(BAR_STEP, CW * 32); // colour c of the tile is complete before anyone reads it
        }
        // ---- epilogue: interior rows were never stored; write them back (boundary rows are current) ----
        for (int i = n_bnd; i < RPW; ++i) {
            const uint4 d = desc[i];
#pragma unroll
            for (int c = 0; c < 2; ++c)
                *(ulonglong2 *)(a.spins + (size_t)c * Nh + d.y + 2 * lane) =
                    *(const ulonglong2 *)((const unsigned char *)(tile + (size_t)c * HZ * HY * Lh) + d.x + 16 * lane);
        }
    }
}

// Host side of the row schedule (see RowTable).  Boundary rows are dealt out along the ring, interior rows along a
// boustrophedon path, so consecutive rows of a warp are lattice neighbours and alternate in (yy + zz) parity.
template <typename G> static bool build_row_table(RowTable<G> &t)
{
    constexpr int TY = G::TY, TZ = G::TZ, CW = G::CW, RPW = G::ROWS / G::CW;
    static_assert(TY % 2 == 0 && TZ % 2 == 0, "tile origin parity must be even");
    std::vector<std::pair<int, int>> ring, snake;
    for (int yy = 1; yy <= TY; ++yy) ring.push_back({yy, 1});
    for (int zz = 2; zz <= TZ; ++zz) ring.push_back({TY, zz});
    for (int yy = TY - 1; yy >= 1; --yy) ring.push_back({yy, TZ});
    for (int zz = TZ - 1; zz >= 2; --zz) ring.push_back({1, zz});
    for (int zz = 2; zz <= TZ - 1; ++zz)
        for (int j = 0; j < TY - 2; ++j) snake.push_back({(zz & 1) ? TY - 1 - j : 2 + j, zz});
    if ((int)ring.size() != G::NB || (int)(ring.size() + snake.size()) != G::ROWS) return false;
    // boundary rows: the first (NB % CW) warps... every warp gets floor or ceil of NB / CW consecutive ring rows
    const int lo = G::NB / CW, n_hi = G::NB % CW; // n_hi warps take lo + 1
    int pos = 0;
    int need[CW], len[CW];
    for (int w = 0; w < CW; ++w) {
        const int nb = lo + (w < n_hi ? 1 : 0);
        t.n_bnd[w] = (uint8_t)nb;
        t.phi[w] = nb ? (uint8_t)((ring[pos].first + ring[pos].second) & 1) : 0;
        for (int i = 0; i < nb; ++i, ++pos) t.row[w][i] = (uint16_t)(ring[pos].first | (ring[pos].second << 8));
        need[w] = (t.phi[w] + nb) & 1; // parity the first interior row must have
        len[w] = RPW - nb;
    }
    // interior rows: walk the snake, each time handing the next segment to a warp whose parity fits
    bool done[CW] = {};
    pos = 0;
    for (int n = 0; n < CW; ++n) {
        int pick = -1;
        for (int w = 0; w < CW && pick < 0; ++w) {
            if (done[w]) continue;
            if (len[w] == 0) pick = w;
            else if (pos < (int)snake.size() && ((snake[pos].first + snake[pos].second) & 1) == need[w]) pick = w;
        }
        if (pick < 0) return false;
        done[pick] = true;
        for (int i = 0; i < len[pick]; ++i, ++pos) {
            if (pos >= (int)snake.size()) return false;
            t.row[pick][t.n_bnd[pick] + i] = (uint16_t)(snake[pos].first | (snake[pos].second << 8));
        }
    }
    if (pos != (int)snake.size()) return false;
    // check: every row once, alternating parity from phi, boundary rows first
    std::vector<int> seen((TY + 2) * (TZ + 2), 0);
    for (int w = 0; w < CW; ++w)
        for (int i = 0; i < RPW; ++i) {
            const int yy = t.row[w][i] & 0xff, zz = t.row[w][i] >> 8;
            const bool isB = yy == 1 || yy == TY || zz == 1 || zz == TZ;
            if (yy < 1 || yy > TY || zz < 1 || zz > TZ || seen[zz * (TY + 2) + yy]++) return false;
            if (((yy + zz) & 1) != ((t.phi[w] + i) & 1) || isB != (i < t.n_bnd[w])) return false;
        }
    return true;
}

// ---------------------------------------------------------------------------------------------
// 32-bit bond words (2 replicas): 16 compute warps of 96 registers.  64-bit bond words: twice the bond registers in
// flight, so 8 compute warps with up to 168 registers each.  Both unroll two row pairs per loop iteration: measured
// best (4.83 / 6.14 us per half-sweep; no unrolling 5.3 / 6.4, full unrolling 4.91 / 9.2 -- instruction cache).
template <typename BondT> struct Geom128Of { typedef ResidentGeom<128, 16, 8, 16, 2> type; };
template <> struct Geom128Of<uint64_t> { typedef ResidentGeom<128, 16, 8, 8, 2> type; };
typedef Geom128Of<uint32_t>::type Geom128; // tile shape, grid and flag layout are the same for both

template <typename BondT, bool ALWAYS, bool RARE, bool HB = false>
static cudaError_t launch_resident_typed(ResidentArgs &a, cudaStream_t st)
{
    typedef typename Geom128Of<BondT>::type G;
    static_assert(G::G == Geom128::G && G::SMEM_BYTES == Geom128::SMEM_BYTES, "one flag / shared-memory layout");
    static RowTable<G> tab;
    static const bool tab_ok = build_row_table<G>(tab);
    if (!tab_ok) return cudaErrorInvalidConfiguration;
    auto kern = k_sweep_resident<G, BondT, ALWAYS, RARE, HB>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    void *args[] = {&a, &tab};
    return cudaLaunchCooperativeKernel((void *)kern, dim3(G::G), dim3(G::THREADS), args, G::SMEM_BYTES, st);
}

bool resident_supported(const ea_sim *s, std::string *why)
{
    auto no = [&](const char *msg) { if (why) *why = msg; return false; };
    if (s->lat.L != 128) return no("resident kernel: L must be 128");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) return no("resident kernel: cudaGetDeviceProperties failed");
    if (!prop.cooperativeLaunch) return no("resident kernel: the device has no cooperative launch");
    if (prop.multiProcessorCount < Geom128::G) return no("resident kernel: the device has fewer than 128 SMs");
    if (prop.sharedMemPerBlockOptin < Geom128::SMEM_BYTES) return no("resident kernel: the device has less than 187 KB of shared memory per CTA");
    return true;
}

// host-only check of the row schedules of both geometries (every row once, boundary rows first, alternating parity)
bool resident_tables_ok()
{
    RowTable<Geom128Of<uint32_t>::type> t32;
    RowTable<Geom128Of<uint64_t>::type> t64;
    return build_row_table<Geom128Of<uint32_t>::type>(t32) && build_row_table<Geom128Of<uint64_t>::type>(t64);
}

size_t resident_flag_bytes() { return (size_t)(Geom128::G * 32 + 32) * sizeof(unsigned); }

// n sweeps starting at sweep index t0, one launch.  Asynchronous; ea_sim::resident_epoch advances by 2n.
cudaError_t launch_sweeps_resident(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st)
{
    ResidentArgs a;
    a.spins = s->spins;
    a.bonds = s->bonds;
    { const SweepRng g0 = make_sweep_rng(s->seed, 0, 0);
      for (int r = 0; r < 10; ++r) { a.k0[r] = g0.k0[r]; a.k1[r] = g0.k1[r]; } }
    a.t0 = t0;
    a.n_half = 2 * n;
    a.epoch0 = s->resident_epoch;
    a.flags = s->resident_flags;
    a.abort_flag = s->resident_flags + Geom128::G * 32;
    a.timeout_ns = s->resident_timeout_ns;
    a.th = s->th;
    const bool always = a.th.always[0] | a.th.always[1] | a.th.always[2];
    // low temperature: energy-raising moves are rare enough for a warp-level branch (see metropolis_word)
    const bool rare = !always && a.th.thr[2] < RARE_THR2_MAX;
    cudaError_t e;
    if (s->dynamics == EA_DYN_HEATBATH) // heat bath (C-HB) carries its own always-masks; no rare branch
        e = s->n_replicas == 2 ? launch_resident_typed<uint32_t, false, false, true>(a, st)
                               : launch_resident_typed<uint64_t, false, false, true>(a, st);
    else if (s->n_replicas == 2)
        e = always ? launch_resident_typed<uint32_t, true, false>(a, st)
            : rare ? launch_resident_typed<uint32_t, false, true>(a, st)
                   : launch_resident_typed<uint32_t, false, false>(a, st);
    else
        e = always ? launch_resident_typed<uint64_t, true, false>(a, st)
            : rare ? launch_resident_typed<uint64_t, false, true>(a, st)
                   : launch_resident_typed<uint64_t, false, false>(a, st);
    if (e == cudaSuccess) {
        s->resident_epoch += 2 * n;
        s->count_launch();
    }
    return e;
}

} // namespace ea

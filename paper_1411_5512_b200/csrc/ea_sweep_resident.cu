// ea_sweep_resident.cu -- RESIDENT: a persistent half-sweep kernel for L = 128 that keeps the whole spin
// lattice in shared memory for the n sweeps of one ea_sweep(n) call.
//
// Same update as every other variant (Eq. 9; checkerboard order PAPER.md:80-86) and the same
// stream contract, hence bit-identical results.  What changes is where the colour barrier ("each
// half-step is performed in its own CUDA kernel call to ensure global synchronization") comes from:
//
//   * the y-z plane of x-rows is cut into rectangular tiles, one CTA per tile, one CTA per SM (cooperative
//     launch: all CTAs are co-resident).  On a 148-SM part: 9 strips of 14 y-rows cut into 16 tiles of 14 x 8 rows
//     (112 rows = 7 per compute warp) plus one strip of 2 y-rows cut into 4 tiles of 2 x 32 rows -- 148 tiles, every
//     SM busy.  (Fewer SMs: 128 tiles of 16 x 8.)  A CTA holds both colours of its rows plus a one-row halo ring in
//     shared memory; only the bond words stream in (from L2: bonds never change).
//   * rows come in two classes by (y + z) parity.  All four neighbour rows of a row are of the OTHER class, so a
//     half-step splits into two phases (class c first, then class 1 - c; the class order flips with the colour)
//     and phase k depends only on phase k - 2 of the other warps and of the neighbouring CTAs.  The barrier a warp
//     waits on was armed a whole phase earlier: nobody idles at a colour boundary, within the CTA (two mbarriers)
//     or across CTAs (boundary rows of a class are updated first and stored to the global array as well; a producer
//     warp publishes "phase k done" (release store of a flag), waits for the same flag of the neighbouring tiles and
//     pulls their fresh boundary rows of that class into the halo ring with 1-D bulk TMA copies).  No grid-wide
//     barrier, no relaunch.
//   * in a phase every row has the same x-phase S = (colour ^ y ^ z) & 1 -- S = 0 in the first phase of every
//     half-step and S = 1 in the second -- so the x-neighbour selection is compile-time.
//   * global memory always holds the current boundary rows; interior rows are written back once at the end,
//     so after the launch the global array is the full state at time t0 + n.
#include <string.h>

#include <utility>
#include <vector>

#include "ea_internal.h"
#include "ea_sweep_common.cuh"

namespace ea {

constexpr int RES_L = 128, RES_LH = RES_L / 2;
constexpr unsigned RES_NH = (unsigned)RES_L * RES_L * RES_L / 2;
constexpr int RES_ROW_BYTES = RES_LH * 8; // one colour of one x-row
constexpr int RES_MAX_CTAS = 160;         // flag lines reserved in the workspace
constexpr int RES_MAX_NB = 12;            // neighbouring tiles of a tile
constexpr int RES_MAX_CP = 36;            // halo rows of one class
constexpr int RES_PRODUCERS = 2;          // producer warps: one for the even phases, one for the odd ones
constexpr int RES_SLOTS = 240;            // row slots per class and CTA: compute warps (8, 16, 20, 24) x rows per warp and class
constexpr int RES_MAX_CW = 24;
constexpr int RES_SMEM_CPL = 128 + 2 * RES_SLOTS * 16;                 // 4 mbarriers (64 B used), then the row descriptors,
constexpr int RES_SMEM_HDR = RES_SMEM_CPL + 2 * 40 * 8;               // then the halo copy list [2][40] (RES_MAX_CP <= 40)
static_assert(RES_SMEM_HDR % 128 == 0 && RES_MAX_CP <= 40, "the tile starts on a 128-byte line");

// One tile = one CTA (host-built, build_partition; lives in the sim's workspace).
struct ResTile {
    uint16_t y0, z0, TY, TZ;     // origin (even) and shape in rows
    uint16_t n_nb, nbp;          // neighbouring tiles; leading row PAIRS of a warp's phase that may hold boundary rows
    uint16_t n_cp[2];            // halo rows per class
    uint16_t nb[RES_MAX_NB];     // CTA indices of the neighbouring tiles
    uint2 cp[2][RES_MAX_CP];     // halo copy: x = word offset of the row in a global colour plane, y = in a tile colour plane
    uint16_t row[2][RES_SLOTS];  // [class][warp * (RES_SLOTS / CW) + slot] = yy | zz << 8 (tile coordinates, from 1)
    uint8_t n_rows[2][RES_MAX_CW]; // [class][warp]: rows of that class, boundary rows first
    uint8_t n_bnd[2][RES_MAX_CW];
};

struct ResidentArgs {
    uint64_t *spins;     // [2][Nh]
    const void *bonds;   // BondT [2][3][Nh]
    const ResTile *tiles;
    uint32_t k0[10], k1[10]; // Philox round keys of the seed (C-A6)
    uint64_t t0;         // first sweep index
    uint32_t n_half;     // half-steps to run (2 per sweep)
    uint32_t epoch0;     // flag value before this launch; phase k publishes epoch0 + k + 1
    unsigned *flags;     // [RES_MAX_CTAS][32]: one 128-byte line per CTA; word 0 / 1 = last even / odd phase published
    unsigned *abort_flag;// set by any CTA whose wait timed out; everybody then leaves
    unsigned long long timeout_ns; // a neighbour that never shows up: give up after this long
    Thresholds th;
#ifdef EA_RES_TRACE
    long long *trace; // [2 tiles][32 warps][8 phases][8 events] SM clocks (debug builds only)
#endif
};

#ifdef EA_RES_TRACE
#define RES_TRACE(a, b, warp, lane, k, ev)                                                                          \
    do {                                                                                                            \
        if ((a).trace && ((b) == 0 || (b) == 144) && (k) >= 200 && (k) < 208 && (lane) == 0)                        \
            (a).trace[((((b) ? 1 : 0) * 32 + (warp)) * 8 + ((k) - 200)) * 8 + (ev)] = clock64();                    \
    } while (0)
#else
#define RES_TRACE(a, b, warp, lane, k, ev) do { } while (0)
#endif

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, unsigned parity)
{
    uint32_t ok;
    // with a suspend-time hint the thread sleeps in hardware until the phase completes (or the hint expires) instead of
    // returning at once: a spinning warp would take issue slots from the warps it is waiting for
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)
                 : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    while (!mbar_try_wait(bar, parity)) { }
}
// 16-byte asynchronous copy global -> shared, L2 only (cp.async.cg = LDGSTS.BYPASS: never served from a stale L1 line)
__device__ __forceinline__ void cp_async16(uint32_t dst_smem, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");
}
// one arrival on the mbarrier once every cp.async this thread has issued so far has landed (the count is not raised:
// the barrier is initialised for one such arrival per lane)
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
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

// Named barriers 1..4, one per phase index mod 4: "the boundary rows of phase k are stored".  Four, not two: a warp without
// boundary rows does not wait for the halo, so it may arrive for phase k + 2 before the producer has consumed the barrier of
// phase k; it cannot arrive for k + 4 before that (phase k + 2 of the boundary warps needs the producer's copies of phase k).
enum { BAR_BOUNDARY0 = 1 };
constexpr uint32_t RARE_THR2_MAX = 0x04000000u; // P(r < thr[2]) < 1/64: the warp-level branch of metropolis_word pays

template <typename BondT> struct RowBonds { typename Pair<BondT>::type jx, jy, jz, bx, by, bz; };

// Row descriptor (shared memory, one per (class, compute warp, row slot), written once in the prologue):
//   x = byte offset of row (zz, yy) inside a colour plane of the tile
//   y = word offset of row (y, z) inside a colour plane of the global arrays, Lh * (y + L * z)
//   z = Nh + offset of row (y-1, z),  w = 2 Nh + offset of row (y, z-1)    (periodic) -- the backward y / z bonds
__device__ __forceinline__ uint4 make_row_desc(unsigned yy, unsigned zz, unsigned y0, unsigned z0, unsigned HY)
{
    constexpr unsigned Lh = RES_LH, L = RES_L, Nh = RES_NH;
    const unsigned y = y0 + yy - 1, z = z0 + zz - 1;
    uint4 d;
    d.x = (zz * HY + yy) * RES_ROW_BYTES;
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
__device__ __forceinline__ RowBonds<BondT> load_row_bonds(const Ptr32 Jc_l, const Ptr32 Jo_l, const uint4 d)
{
    constexpr unsigned Nh = RES_NH;
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
    uint32_t s_own, s_oth;   // shared-memory address of the tile plane of colour c / 1 - c, + 16 * lane
    uint32_t planeb;         // bytes between z-planes of the tile (CTA-uniform)
    Ptr32 g_own;             // global plane of colour c + 2 * lane
    Ptr32 Jc_l, Jo_l;        // bond planes of colour c / 1 - c + 2 * lane
    unsigned k;
    int lane_m, lane_p;
#ifdef EA_RES_TRACE
    long long *trace; unsigned tb, tw, tk; // debug builds: trace buffer, CTA, warp, phase
#endif
};

// shared-memory accesses by 32-bit shared address (one IADD per row address instead of generic pointer arithmetic:
// measured 4.34 against 4.41 us per half-sweep)
__device__ __forceinline__ ulonglong2 lds128(uint32_t addr)
{
    ulonglong2 v;
    asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, ulonglong2 v)
{
    asm volatile("st.shared.v2.u64 [%0], {%1, %2};" ::"r"(addr), "l"(v.x), "l"(v.y) : "memory");
}

__device__ __forceinline__ void stg128(void *p, ulonglong2 v)
{
    // volatile keeps it (no outputs) and in order with the barrier arrive that follows; no memory clobber: the rows around it
    // stay free to interleave
    asm volatile("st.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(v.x), "l"(v.y));
}

// the four random numbers of the lane's two words of a row (d.y = row offset, S = row phase; C-A7): independent of the
// spins, so they are drawn one row ahead and their IMAD.WIDE chain (fma pipe) overlaps the LOP3 logic (alu pipe)
// of the row before
__device__ __forceinline__ uint4 row_random(const SweepRng &g, const unsigned k, const unsigned S, const uint4 d)
{
    // canonical site = x + L (y + L z), L = 2 Lh; the lane's two words (xh = 2k, 2k + 1) are one pair: one block
    return sweep_random4(g, 4 * k + S + 2 * d.y);
}

// one row of colour c with compile-time phase S; publishes it to global when `publish`
template <int S, typename BondT, bool ALWAYS, bool RARE, bool HB>
__device__ __forceinline__ void resident_row(const ResidentStep &x, const uint4 d, const RowBonds<BondT> &bd,
                                             const uint4 r, const Thresholds &th, const bool publish)
{
    const uint32_t own_row = x.s_own + d.x, o = x.s_oth + d.x;
    const ulonglong2 own = lds128(own_row);
    const ulonglong2 P0 = lds128(o);
    const ulonglong2 Pm = lds128(o - RES_ROW_BYTES);
    const ulonglong2 Pp = lds128(o + RES_ROW_BYTES);
    const ulonglong2 Zm = lds128(o - x.planeb);
    const ulonglong2 Zp = lds128(o + x.planeb);
    const ulonglong2 out = update_pair_r<S, BondT, ALWAYS, RARE, HB>(own, P0, Pm, Pp, Zm, Zp, bd.jx, bd.jy, bd.jz, bd.bx, bd.by,
                                                                     bd.bz, r, th, x.lane_m, x.lane_p);
    sts128(own_row, out);
    if (publish) stg128(x.g_own.at<ulonglong2>(d.y / 2), out);
}

// One phase of one compute warp: its n rows of one class (all of x-phase S), boundary rows first (nb of them, inside
// the first nbp pairs).  Carried across rows, phases and steps: nxt = bond words of the next row, rnx = its random
// numbers.  dnext / xn / gn describe the first row of the NEXT phase (x-phase 1 - S).
template <int S, typename BondT, bool ALWAYS, bool RARE, bool HB>
__device__ __forceinline__ void resident_phase(const ResidentStep &x, const uint4 *__restrict__ desc, const int n, const int nb,
                                               const int nbp, const int bar_id, const int bar_threads,
                                               RowBonds<BondT> &nxt, uint4 &rnx, const SweepRng &g, const uint4 dnext,
                                               const Ptr32 Jc_next, const Ptr32 Jo_next, const SweepRng &gn,
                                               const Thresholds &th)
{
    const int npairs = n >> 1;
    bool arrived = false;
    if (nb == 0) { // no boundary rows in this phase: nothing of this warp for the producer to wait for
        named_bar_arrive(bar_id, bar_threads);
        arrived = true;
    }
#ifdef EA_RES_VAR_UNROLL2
#pragma unroll 2
#else
#pragma unroll 1
#endif
    for (int j = 0; j < npairs; ++j) {
        const int i = 2 * j;
        const bool last = i + 2 >= n;
        const uint4 d0 = desc[i], d1 = desc[i + 1];
        const uint4 d2 = last ? dnext : desc[i + 2];
        const RowBonds<BondT> b0 = nxt;
        const uint4 r0 = rnx;
        const RowBonds<BondT> b1 = load_row_bonds<BondT>(x.Jc_l, x.Jo_l, d1);
        const uint4 r1 = row_random(g, x.k, S, d1);
        resident_row<S, BondT, ALWAYS, RARE, HB>(x, d0, b0, r0, th, i < nb);
        // the row after next; after the last row of the phase that is the first row of the next phase: other x-phase,
        // and (across a half-step) the colours swap roles and the stream moves on
        if (!last) {
            nxt = load_row_bonds<BondT>(x.Jc_l, x.Jo_l, d2);
            rnx = row_random(g, x.k, S, d2);
        } else {
            nxt = load_row_bonds<BondT>(Jc_next, Jo_next, d2);
            rnx = row_random(gn, x.k, 1 - S, d2);
        }
        resident_row<S, BondT, ALWAYS, RARE, HB>(x, d1, b1, r1, th, i + 1 < nb);
        if (j == nbp - 1 && !arrived) { // every boundary row of this warp and phase is stored (an asm statement is a scheduling fence:
            named_bar_arrive(bar_id, bar_threads); // it sits where a loop trip ends anyway)
            arrived = true;
#ifdef EA_RES_TRACE
            if (x.trace && (x.tb == 0 || x.tb == 144) && x.tk >= 200 && x.tk < 208 && x.k == 0)
                x.trace[(((x.tb ? 1 : 0) * 32 + x.tw) * 8 + (x.tk - 200)) * 8 + 3] = clock64();
#endif
        }
    }
    if (n & 1) {
        const uint4 d0 = desc[n - 1];
        const RowBonds<BondT> b0 = nxt;
        const uint4 r0 = rnx;
        nxt = load_row_bonds<BondT>(Jc_next, Jo_next, dnext);
        rnx = row_random(gn, x.k, 1 - S, dnext);
        resident_row<S, BondT, ALWAYS, RARE, HB>(x, d0, b0, r0, th, n - 1 < nb);
    }
    if (!arrived) named_bar_arrive(bar_id, bar_threads);
}

template <int CW, typename BondT, bool ALWAYS, bool RARE, bool HB>
__global__ void __launch_bounds__((CW + RES_PRODUCERS) * 32, 1) k_sweep_resident(const ResidentArgs a)
{
    constexpr int L = RES_L, Lh = RES_LH, THREADS = (CW + RES_PRODUCERS) * 32, RPC = RES_SLOTS / CW;
    constexpr int BAR_THREADS = (CW + 1) * 32; // a boundary barrier: every compute warp arrives, one producer warp waits
    constexpr unsigned Nh = RES_NH;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *phase_bar = (uint64_t *)smem_raw;        // [2]: phase k of every compute warp is complete (k & 1)
    uint64_t *halo_bar = (uint64_t *)(smem_raw + 16);  // [2]: the halo rows written in phase k have landed (k & 1)
    uint4 *rowdesc = (uint4 *)(smem_raw + 128);        // [2][RES_SLOTS] row descriptors
    uint2 *cpl = (uint2 *)(smem_raw + RES_SMEM_CPL);   // [2][40] halo copies of each class: byte offsets (global row, tile row) in a colour plane
    uint64_t *tile = (uint64_t *)(smem_raw + RES_SMEM_HDR); // [2][HZ][HY][Lh]

    const unsigned tid = threadIdx.x, lane = tid & 31;
    const unsigned warp = __shfl_sync(0xffffffffu, tid >> 5, 0); // provably warp-uniform: no divergence guards around the shuffles
    const unsigned b = blockIdx.x;
    const ResTile *__restrict__ T = a.tiles + b;
    const unsigned y0 = __ldg(&T->y0), z0 = __ldg(&T->z0), TY = __ldg(&T->TY), TZ = __ldg(&T->TZ);
    const unsigned HY = TY + 2, HZ = TZ + 2;
    const unsigned plane_words = HZ * HY * Lh; // one colour of the tile with its halo ring
    const uint32_t n_phases = 2 * a.n_half;

    // ---- prologue: barriers, row descriptors, tile + halo ring of both colours from global ---------------
    for (unsigned v = tid; v < 2u * RES_SLOTS; v += THREADS) {
        const unsigned code = __ldg(&T->row[0][0] + v);
        rowdesc[v] = make_row_desc(code & 0xff, code >> 8, y0, z0, HY);
    }
    for (unsigned v = tid; v < 2u * 40; v += THREADS) { // padded with repeats of the last entry: the producer copies four per trip
        const unsigned cls = v / 40, i = v % 40, n = __ldg(&T->n_cp[cls]);
        const uint2 e = __ldg(&T->cp[cls][i < n ? i : n - 1]);
        cpl[v] = make_uint2(e.x * 8, e.y * 8); // byte offsets
    }
    if (tid == 0) {
        mbar_init(phase_bar + 0, CW);
        mbar_init(phase_bar + 1, CW);
        mbar_init(halo_bar + 0, 32); // one arrival per lane of the producer warp, when its copies have landed
        mbar_init(halo_bar + 1, 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (unsigned v = tid; v < 2u * HZ * HY * (Lh / 2); v += THREADS) {
        const unsigned w2 = v % (Lh / 2), r = v / (Lh / 2);
        const unsigned yy = r % HY, zz = (r / HY) % HZ, c = r / (HY * HZ);
        const unsigned y = (y0 + yy - 1) & (L - 1), z = (z0 + zz - 1) & (L - 1);
        const ulonglong2 val = *(const ulonglong2 *)(a.spins + (size_t)c * Nh + Lh * (y + L * z) + 2 * w2);
        *(ulonglong2 *)(tile + (size_t)c * plane_words + (size_t)(zz * HY + yy) * Lh + 2 * w2) = val;
    }
    __syncthreads();

    const BondT *__restrict__ bonds = (const BondT *)a.bonds;

    if (warp >= (unsigned)CW) {
        // ---- producer warps: publish our boundary rows, fetch the neighbours'.  Warp CW serves the even phases, warp
        // CW + 1 the odd ones (own flag word, own barriers), so the latency chain of one phase -- release, the
        // neighbours' release becoming visible, issuing the copies -- overlaps that of the next ------------------------
        const unsigned n_nb = __ldg(&T->n_nb);
        const unsigned nb_tile = lane < n_nb ? __ldg(&T->nb[lane]) : 0;
        const unsigned n_cp0 = __ldg(&T->n_cp[0]), n_cp1 = __ldg(&T->n_cp[1]);
        for (uint32_t k = warp - CW; k < n_phases; k += RES_PRODUCERS) {
            const unsigned c = (k >> 1) & 1, cls = c ^ (k & 1); // phase k updates colour c of the rows of class cls
            RES_TRACE(a, b, warp, lane, k, 0);
            named_bar_sync(BAR_BOUNDARY0 + (k & 3), BAR_THREADS);   // its boundary rows are in smem and in global
            RES_TRACE(a, b, warp, lane, k, 1);
            const unsigned epoch = a.epoch0 + k + 1;
#ifdef EA_RES_TRACE
            { // the barrier blocks at the first access to barrier-protected state, not at its issue: make one, then stamp
                unsigned dummy;
                asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(dummy) : "r"(smem_u32(phase_bar)) : "memory");
                if (a.trace && (b == 0 || b == 144) && k >= 200 && k < 208 && lane == 0)
                    a.trace[((((b) ? 1 : 0) * 32 + warp) * 8 + (k - 200)) * 8 + 5] = clock64() + (dummy & 0);
                if (lane == 0) asm volatile("fence.acq_rel.gpu;" ::: "memory");
                RES_TRACE(a, b, warp, lane, k, 6);
            }
#endif
            if (lane == 0) st_release_gpu(a.flags + b * 32 + (k & 1), epoch); // release: cumulative over the CTA's stores
            RES_TRACE(a, b, warp, lane, k, 4);
            if (k + 2 >= n_phases) continue;                    // nobody reads the halo of the last two phases
            bool ok = true;
            if (lane < n_nb) {
                const unsigned *f = a.flags + nb_tile * 32 + (k & 1);
                const unsigned long long t_start = globaltimer_ns();
                unsigned spins = 0;
                while ((int)(ld_acquire_gpu(f) - epoch) < 0) {
                    __nanosleep(64); // the poll must not compete with the compute warps for issue slots
                    if ((++spins & 63u) == 0) {
                        if (*(volatile unsigned *)a.abort_flag || globaltimer_ns() - t_start > a.timeout_ns) {
                            ok = false;
                            break;
                        }
                    }
                }
            }
            ok = __all_sync(0xffffffffu, ok);
            RES_TRACE(a, b, warp, lane, k, 2);
            // on a time-out: raise the abort flag (every CTA stops waiting), keep going with stale halos so that
            // all barriers still complete; the host finds the flag at its next synchronisation and reports it
            if (!ok && lane == 0) atomicExch(a.abort_flag, 1u);
            // one 512-byte row per warp instruction (16 bytes per lane), all in flight together; the barrier of this phase
            // parity completes when every lane's copies have landed
            const unsigned ncp = cls ? n_cp1 : n_cp0;
            const uint2 *list = cpl + cls * 40;
            const uint32_t dst = smem_u32(tile) + c * plane_words * 8 + 16 * lane;
            const Ptr32 src(a.spins + (size_t)c * Nh + 2 * lane);
            for (unsigned i = 0; i < ncp; i += 4) { // the list is padded to a multiple of four with repeats of its last entry
                const uint4 e01 = *(const uint4 *)(list + i), e23 = *(const uint4 *)(list + i + 2);
                cp_async16(dst + e01.y, src.at<const char>(e01.x));
                cp_async16(dst + e01.w, src.at<const char>(e01.z));
                cp_async16(dst + e23.y, src.at<const char>(e23.x));
                cp_async16(dst + e23.w, src.at<const char>(e23.z));
            }
            cp_async_arrive_noinc(halo_bar + (k & 1));
            RES_TRACE(a, b, warp, lane, k, 3);
        }
    } else {
        // ---- compute warps -----------------------------------------------------------------------------
        const int n_rows0 = __ldg(&T->n_rows[0][warp]), n_rows1 = __ldg(&T->n_rows[1][warp]);
        const int n_bnd0 = __ldg(&T->n_bnd[0][warp]), n_bnd1 = __ldg(&T->n_bnd[1][warp]);
        const int nbp = __ldg(&T->nbp);
        const uint4 *__restrict__ desc0 = rowdesc + warp * RPC;             // rows of class 0
        const uint4 *__restrict__ desc1 = rowdesc + RES_SLOTS + warp * RPC; // rows of class 1
        const uint4 first0 = desc0[0], first1 = desc1[0];
        ResidentStep x;
        x.k = lane;
        x.lane_m = (int)((lane - 1) & 31);
        x.lane_p = (int)((lane + 1) & 31);
        x.planeb = HY * RES_ROW_BYTES;
        const uint32_t tile_s = smem_u32(tile) + 16 * lane, plane_bytes = plane_words * 8;
        SweepRng g;
#pragma unroll
        for (int r = 0; r < 10; ++r) { g.k0[r] = a.k0[r]; g.k1[r] = a.k1[r]; }
        const Ptr32 J0_l(bonds + 2 * lane), J1_l(bonds + (size_t)3 * Nh + 2 * lane);

        // software pipeline: the bond words and the random numbers of the next row are always in flight.
        // Phase 0 = colour 0, class 0, x-phase 0.
        RowBonds<BondT> nxt = load_row_bonds<BondT>(J0_l, J1_l, first0);
        sweep_rng_set_time(g, a.t0, 0u);
        uint4 rnx = row_random(g, lane, 0u, first0);
        for (uint32_t h = 0; h < a.n_half; ++h) {
            const unsigned c = h & 1;
            sweep_rng_set_time(g, a.t0 + (h >> 1), c);
            SweepRng gn = g;
            sweep_rng_set_time(gn, a.t0 + ((h + 1) >> 1), 1 - c);
            x.Jc_l = c ? J1_l : J0_l;
            x.Jo_l = c ? J0_l : J1_l;
            x.s_own = tile_s + c * plane_bytes;
            x.s_oth = tile_s + (1 - c) * plane_bytes;
            x.g_own = Ptr32(a.spins + (size_t)c * Nh + 2 * lane);
            // keep the per-step bases in registers: recomputing them from c inside the row loop costs alu-pipe selects
            asm volatile("" : "+l"(x.Jc_l.base), "+l"(x.Jo_l.base), "+l"(x.g_own.base), "+r"(x.s_own), "+r"(x.s_oth));
            const unsigned par = (h - 1) & 1; // phase k waits for generation (k >> 1) - 1 = h - 1 of barrier k & 1
            // first phase of the half-step: rows of class c (x-phase 0); then class 1 - c (x-phase 1).  Phase k = 2h, 2h + 1
            // needs phase k - 2 of every warp of the CTA and the halo rows the neighbours wrote in their phase k - 2.
            RES_TRACE(a, b, warp, lane, 2 * h, 0);
            // (only boundary rows read the halo ring: a warp without any in this phase does not wait for it)
            if (h > 0) { mbar_wait(phase_bar + 0, par); RES_TRACE(a, b, warp, lane, 2 * h, 1); if (c ? n_bnd1 : n_bnd0) mbar_wait(halo_bar + 0, par); }
            RES_TRACE(a, b, warp, lane, 2 * h, 2);
#ifdef EA_RES_TRACE
            x.trace = a.trace; x.tb = b; x.tw = warp; x.tk = 2 * h;
#endif
            resident_phase<0, BondT, ALWAYS, RARE, HB>(x, c ? desc1 : desc0, c ? n_rows1 : n_rows0, c ? n_bnd1 : n_bnd0, nbp,
                                                        BAR_BOUNDARY0 + ((2 * h) & 3), BAR_THREADS, nxt, rnx, g, c ? first0 : first1, x.Jc_l, x.Jo_l, g, a.th);
            __syncwarp();
            if (lane == 0) mbar_arrive(phase_bar + 0);
            RES_TRACE(a, b, warp, lane, 2 * h, 4);
            RES_TRACE(a, b, warp, lane, 2 * h + 1, 0);
            if (h > 0) { mbar_wait(phase_bar + 1, par); RES_TRACE(a, b, warp, lane, 2 * h + 1, 1); if (c ? n_bnd0 : n_bnd1) mbar_wait(halo_bar + 1, par); }
            RES_TRACE(a, b, warp, lane, 2 * h + 1, 2);
#ifdef EA_RES_TRACE
            x.tk = 2 * h + 1;
#endif
            // the next phase is the first of half-step h + 1: colour 1 - c, class 1 - c -- the class just done
            resident_phase<1, BondT, ALWAYS, RARE, HB>(x, c ? desc0 : desc1, c ? n_rows0 : n_rows1, c ? n_bnd0 : n_bnd1, nbp,
                                                        BAR_BOUNDARY0 + ((2 * h + 1) & 3), BAR_THREADS, nxt, rnx, g, c ? first0 : first1, x.Jo_l, x.Jc_l, gn, a.th);
            __syncwarp();
            if (lane == 0) mbar_arrive(phase_bar + 1);
            RES_TRACE(a, b, warp, lane, 2 * h + 1, 4);
        }
        // ---- epilogue: interior rows were never stored; write them back (boundary rows are current) ----
        // (rows of this warp only: nobody else writes them, and this warp's last writes are in program order)
#pragma unroll
        for (int cls = 0; cls < 2; ++cls) {
            const uint4 *desc = cls ? desc1 : desc0;
            const int n = cls ? n_rows1 : n_rows0, nb = cls ? n_bnd1 : n_bnd0;
            for (int i = nb; i < n; ++i) {
                const uint4 d = desc[i];
#pragma unroll
                for (int c = 0; c < 2; ++c)
                    *(ulonglong2 *)(a.spins + (size_t)c * Nh + d.y + 2 * lane) = lds128(tile_s + c * plane_bytes + d.x);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Host side: the partition of the 128 x 128 rows into tiles, and the schedule of every tile.
// ---------------------------------------------------------------------------------------------
struct Rect { int y0, z0, TY, TZ; };

// 148 tiles (every SM of a B200): 9 strips of 14 y-rows x 16 tiles of 8 z-planes (112 rows each: 7 per compute warp)
// + the last 2 y-rows in 4 tiles of 32 z-planes.  Otherwise 128 tiles of 16 x 8.
static std::vector<Rect> make_partition(int n_tiles)
{
    std::vector<Rect> r;
    if (n_tiles == 148) {
        for (int s = 0; s < 9; ++s)
            for (int t = 0; t < 16; ++t) r.push_back({14 * s, 8 * t, 14, 8});
        for (int t = 0; t < 4; ++t) r.push_back({126, 32 * t, 2, 32});
    } else if (n_tiles == 128) {
        for (int s = 0; s < 8; ++s)
            for (int t = 0; t < 16; ++t) r.push_back({16 * s, 8 * t, 16, 8});
    }
    return r;
}

size_t resident_smem_bytes(int n_tiles)
{
    size_t m = 0;
    for (const Rect &q : make_partition(n_tiles)) {
        const size_t s = (size_t)2 * (q.TY + 2) * (q.TZ + 2) * RES_ROW_BYTES;
        if (s > m) m = s;
    }
    return m + RES_SMEM_HDR;
}

// Schedules of all tiles for `cw` compute warps.  Rows of a class are dealt to the warps round-robin, boundary rows
// first; class 1 continues where class 0 stopped, so the totals of the warps differ by at most one row.  Returns false
// (and says why) if a limit of the kernel is exceeded or the self-check fails.
static bool build_partition(int n_tiles, int cw, std::vector<ResTile> &out, std::string *why)
{
    auto no = [&](const char *m) { if (why) *why = m; return false; };
    const std::vector<Rect> rect = make_partition(n_tiles);
    if (rect.empty() || (int)rect.size() != n_tiles || n_tiles > RES_MAX_CTAS) return no("resident kernel: no partition for this number of tiles");
    if (cw < 1 || cw > RES_MAX_CW || RES_SLOTS % cw) return no("resident kernel: bad number of compute warps");
    const int L = RES_L, rpc = RES_SLOTS / cw;
    std::vector<int> owner((size_t)L * L, -1);
    for (int t = 0; t < n_tiles; ++t) {
        const Rect &q = rect[t];
        if ((q.y0 | q.z0 | q.TY | q.TZ) & 1) return no("resident kernel: tile origin and shape must be even");
        for (int z = q.z0; z < q.z0 + q.TZ; ++z)
            for (int y = q.y0; y < q.y0 + q.TY; ++y) {
                if (y >= L || z >= L || owner[(size_t)z * L + y] != -1) return no("resident kernel: tiles overlap");
                owner[(size_t)z * L + y] = t;
            }
    }
    for (int v : owner) if (v < 0) return no("resident kernel: tiles do not cover the lattice");
    out.assign(n_tiles, ResTile());
    for (int t = 0; t < n_tiles; ++t) {
        const Rect &q = rect[t];
        ResTile &T = out[t];
        memset(&T, 0, sizeof(T));
        const int HY = q.TY + 2;
        T.y0 = (uint16_t)q.y0; T.z0 = (uint16_t)q.z0; T.TY = (uint16_t)q.TY; T.TZ = (uint16_t)q.TZ;
        // halo ring (no corners): who owns it, and the copy that refreshes it
        std::vector<int> nbs;
        for (int zz = 0; zz <= q.TZ + 1; ++zz)
            for (int yy = 0; yy <= q.TY + 1; ++yy) {
                const bool ey = yy == 0 || yy == q.TY + 1, ez = zz == 0 || zz == q.TZ + 1;
                if (ey == ez) continue; // interior or corner
                const int y = (q.y0 + yy - 1 + L) % L, z = (q.z0 + zz - 1 + L) % L;
                const int o = owner[(size_t)z * L + y];
                if (o == t) return no("resident kernel: a tile is its own neighbour");
                bool seen = false;
                for (int v : nbs) seen |= v == o;
                if (!seen) nbs.push_back(o);
                const int cls = (yy + zz) & 1;
                if (T.n_cp[cls] >= RES_MAX_CP) return no("resident kernel: too many halo rows");
                T.cp[cls][T.n_cp[cls]++] = make_uint2((unsigned)(RES_LH * (y + L * z)), (unsigned)((zz * HY + yy) * RES_LH));
            }
        if ((int)nbs.size() > RES_MAX_NB) return no("resident kernel: too many neighbouring tiles");
        T.n_nb = (uint16_t)nbs.size();
        for (size_t i = 0; i < nbs.size(); ++i) T.nb[i] = (uint16_t)nbs[i];
        // Rows by class.  The sub-partition schedulers favour the warps with the highest index, which therefore run
        // ahead of the others inside a phase: boundary rows are dealt to the warps from the top down (they are published
        // soonest), interior rows fill the warps up from the bottom so that the totals differ by at most one row.
        int total[RES_MAX_CW] = {0};
        int max_bnd = 0;
        for (int cls = 0; cls < 2; ++cls) {
            std::vector<std::pair<int, int>> rows[2]; // [0] boundary, [1] interior
            for (int zz = 1; zz <= q.TZ; ++zz)
                for (int yy = 1; yy <= q.TY; ++yy) {
                    if (((yy + zz) & 1) != cls) continue;
                    const bool bnd = yy == 1 || yy == q.TY || zz == 1 || zz == q.TZ;
                    rows[bnd ? 0 : 1].push_back({yy, zz});
                }
            const int n_cls = (int)(rows[0].size() + rows[1].size());
            // quota of each warp in this class: floor or ceil of n_cls / cw, the warps with the smaller total so far get the ceil
            int quota[RES_MAX_CW];
            for (int w = 0; w < cw; ++w) quota[w] = n_cls / cw;
            for (int extra = n_cls % cw; extra > 0; --extra) {
                int best = -1;
                for (int w = 0; w < cw; ++w)
                    if (quota[w] == n_cls / cw && (best < 0 || total[w] < total[best])) best = w;
                ++quota[best];
            }
            auto give = [&](int w, const std::pair<int, int> &yz, bool bnd) {
                uint8_t &n = T.n_rows[cls][w];
                T.row[cls][w * rpc + n] = (uint16_t)(yz.first | (yz.second << 8));
                ++n;
                ++total[w];
                if (bnd) { T.n_bnd[cls][w] = n; if (n > max_bnd) max_bnd = n; }
            };
            for (int w = 0; w < cw; ++w) if (quota[w] > rpc - 2) return no("resident kernel: too many rows per warp");
            // boundary rows: top warps first, two each (one row pair), as far as the quotas allow; further passes if rows remain
            size_t bpos = 0;
            for (int pass = 0; pass < rpc && bpos < rows[0].size(); ++pass)
                for (int w = cw - 1; w >= 0 && bpos < rows[0].size(); --w)
                    for (int i = 0; i < 2 && bpos < rows[0].size() && T.n_rows[cls][w] < quota[w]; ++i) give(w, rows[0][bpos++], true);
            if (bpos != rows[0].size()) return no("resident kernel: no room for the boundary rows");
            // interior rows: fill every warp up to its quota
            size_t pos = 0;
            for (int ww = 0; ww < cw; ++ww)
                while (T.n_rows[cls][ww] < quota[ww] && pos < rows[1].size()) give(ww, rows[1][pos++], false);
            if (pos != rows[1].size()) return no("resident kernel: rows left over");
        }
        T.nbp = (uint16_t)((max_bnd + 1) / 2 > 0 ? (max_bnd + 1) / 2 : 1);
        // self-check: every row once, in its class, boundary rows first; every warp has work in both classes
        std::vector<int> seen((size_t)(q.TY + 2) * (q.TZ + 2), 0);
        int lo = 1 << 30, hi = 0;
        for (int ww = 0; ww < cw; ++ww) {
            const int tot = T.n_rows[0][ww] + T.n_rows[1][ww];
            lo = tot < lo ? tot : lo;
            hi = tot > hi ? tot : hi;
            for (int cls = 0; cls < 2; ++cls) {
                if (T.n_rows[cls][ww] < 1) return no("resident kernel: a warp without rows in a class");
                if (T.n_bnd[cls][ww] > 2 * T.nbp) return no("resident kernel: boundary rows beyond the leading pairs");
                for (int i = 0; i < T.n_rows[cls][ww]; ++i) {
                    const int code = T.row[cls][ww * rpc + i], yy = code & 0xff, zz = code >> 8;
                    if (yy < 1 || yy > q.TY || zz < 1 || zz > q.TZ || ((yy + zz) & 1) != cls) return no("resident kernel: bad row in the schedule");
                    if (seen[(size_t)zz * HY + yy]++) return no("resident kernel: a row is scheduled twice");
                    const bool bnd = yy == 1 || yy == q.TY || zz == 1 || zz == q.TZ;
                    if (bnd != (i < T.n_bnd[cls][ww])) return no("resident kernel: boundary rows are not first");
                }
            }
        }
        for (int zz = 1; zz <= q.TZ; ++zz)
            for (int yy = 1; yy <= q.TY; ++yy)
                if (seen[(size_t)zz * HY + yy] != 1) return no("resident kernel: a row is not scheduled");
        if (hi - lo > 1) return no("resident kernel: unbalanced schedule");
    }
    return true;
}

// ---------------------------------------------------------------------------------------------
// 32-bit bond words (2 replicas): 16 compute warps.  64-bit bond words: twice the bond registers in flight, so 8
// compute warps with up to 168 registers each.
template <typename BondT> struct ResidentWarps { static constexpr int CW = 16; };
template <> struct ResidentWarps<uint64_t> { static constexpr int CW = 8; };

static int resident_tiles_for(int n_sm) { return n_sm >= 148 ? 148 : n_sm >= 128 ? 128 : 0; }

template <int CW, typename BondT, bool ALWAYS, bool RARE, bool HB>
static cudaError_t launch_resident_cw(ResidentArgs &a, int n_tiles, cudaStream_t st)
{
    auto kern = k_sweep_resident<CW, BondT, ALWAYS, RARE, HB>;
    const size_t smem = resident_smem_bytes(n_tiles);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    void *args[] = {&a};
    return cudaLaunchCooperativeKernel((void *)kern, dim3(n_tiles), dim3((CW + RES_PRODUCERS) * 32), args, smem, st);
}

static int resident_cw(int n_replicas)
{
    int cw = n_replicas == 2 ? ResidentWarps<uint32_t>::CW : ResidentWarps<uint64_t>::CW;
#ifdef EA_RES_EXPERIMENT
    if (const char *f = getenv("EA_RESIDENT_CW")) cw = atoi(f);
#endif
    return cw;
}

template <typename BondT, bool ALWAYS, bool RARE, bool HB = false>
static cudaError_t launch_resident_typed(ResidentArgs &a, int n_tiles, int cw, cudaStream_t st)
{
#ifdef EA_RES_EXPERIMENT
    if (cw == 12) return launch_resident_cw<12, BondT, ALWAYS, RARE, HB>(a, n_tiles, st);
    if (cw == 20) return launch_resident_cw<20, BondT, ALWAYS, RARE, HB>(a, n_tiles, st);
    if (cw == 24) return launch_resident_cw<24, BondT, ALWAYS, RARE, HB>(a, n_tiles, st);
    if (cw == 16) return launch_resident_cw<16, BondT, ALWAYS, RARE, HB>(a, n_tiles, st);
#endif
    (void)cw;
    return launch_resident_cw<ResidentWarps<BondT>::CW, BondT, ALWAYS, RARE, HB>(a, n_tiles, st);
}

bool resident_supported(const ea_sim *s, std::string *why)
{
    auto no = [&](const char *msg) { if (why) *why = msg; return false; };
    if (s->lat.L != 128) return no("resident kernel: L must be 128");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) return no("resident kernel: cudaGetDeviceProperties failed");
    if (!prop.cooperativeLaunch) return no("resident kernel: the device has no cooperative launch");
    const int n_tiles = resident_tiles_for(prop.multiProcessorCount);
    if (!n_tiles) return no("resident kernel: the device has fewer than 128 SMs");
    if (prop.sharedMemPerBlockOptin < resident_smem_bytes(n_tiles)) return no("resident kernel: the device has too little shared memory per CTA");
    return true;
}

// host-only check of the schedules of both partitions and both warp counts
bool resident_tables_ok()
{
    std::vector<ResTile> t;
    for (int n_tiles : {148, 128})
        for (int cw : {24, 20, 16, 12, 8})
            if (!build_partition(n_tiles, cw, t, nullptr)) return false;
    return true;
}

// flag lines + abort line, then the tile table
size_t resident_flag_bytes() { return (size_t)(RES_MAX_CTAS * 32 + 32) * sizeof(unsigned); }
size_t resident_aux_bytes() { return resident_flag_bytes() + (size_t)RES_MAX_CTAS * sizeof(ResTile); }

// Build the tile table of this sim's device and bond width and put it behind the flags (stream-ordered).
cudaError_t resident_prepare(ea_sim *s, std::string *why)
{
    int n_sm = 0;
    cudaError_t e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, s->device);
    if (e != cudaSuccess) return e;
    if (const char *f = getenv("EA_RESIDENT_TILES")) n_sm = atoi(f) < n_sm ? atoi(f) : n_sm; // tests: force the 128-tile partition
    const int n_tiles = resident_tiles_for(n_sm);
    const int cw = resident_cw(s->n_replicas);
    std::vector<ResTile> t;
    if (!n_tiles || !build_partition(n_tiles, cw, t, why)) return cudaErrorInvalidConfiguration;
    s->resident_tiles = n_tiles;
    // pageable source: staged before the call returns
    return cudaMemcpyAsync((char *)s->resident_flags + resident_flag_bytes(), t.data(), t.size() * sizeof(ResTile),
                           cudaMemcpyHostToDevice, s->stream);
}

#ifdef EA_RES_TRACE
long long *resident_trace_ptr = nullptr;
extern "C" int ea_debug_resident_trace(long long *host) // copies the trace of the last launch (after a sync)
{
    return resident_trace_ptr && cudaMemcpy(host, resident_trace_ptr, 2 * 32 * 8 * 8 * sizeof(long long), cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : 1;
}
#endif

// n sweeps starting at sweep index t0, one launch.  Asynchronous; ea_sim::resident_epoch advances by 4n (two phases
// per half-sweep).
cudaError_t launch_sweeps_resident(ea_sim *s, uint64_t t0, uint32_t n, cudaStream_t st)
{
    if (!s->resident_tiles) return cudaErrorInvalidConfiguration;
    ResidentArgs a;
    a.spins = s->spins;
    a.bonds = s->bonds;
    a.tiles = (const ResTile *)((const char *)s->resident_flags + resident_flag_bytes());
    { const SweepRng g0 = make_sweep_rng(s->seed, 0, 0);
      for (int r = 0; r < 10; ++r) { a.k0[r] = g0.k0[r]; a.k1[r] = g0.k1[r]; } }
    a.t0 = t0;
    a.n_half = 2 * n;
    a.epoch0 = s->resident_epoch;
    a.flags = s->resident_flags;
    a.abort_flag = s->resident_flags + RES_MAX_CTAS * 32;
    a.timeout_ns = s->resident_timeout_ns;
    a.th = s->th;
#ifdef EA_RES_TRACE
    static long long *d_trace = nullptr;
    if (!d_trace) { cudaMalloc(&d_trace, 2 * 32 * 8 * 8 * sizeof(long long)); }
    cudaMemsetAsync(d_trace, 0, 2 * 32 * 8 * 8 * sizeof(long long), st);
    a.trace = d_trace;
    resident_trace_ptr = d_trace;
#endif
    const int nt = s->resident_tiles, cw = resident_cw(s->n_replicas);
    const bool always = a.th.always[0] | a.th.always[1] | a.th.always[2];
    // low temperature: energy-raising moves are rare enough for a warp-level branch (see metropolis_word)
    const bool rare = !always && a.th.thr[2] < RARE_THR2_MAX;
    cudaError_t e;
    if (s->dynamics == EA_DYN_HEATBATH) // heat bath (C-HB) carries its own always-masks; no rare branch
        e = s->n_replicas == 2 ? launch_resident_typed<uint32_t, false, false, true>(a, nt, cw, st)
                               : launch_resident_typed<uint64_t, false, false, true>(a, nt, cw, st);
    else if (s->n_replicas == 2)
        e = always ? launch_resident_typed<uint32_t, true, false>(a, nt, cw, st)
            : rare ? launch_resident_typed<uint32_t, false, true>(a, nt, cw, st)
                   : launch_resident_typed<uint32_t, false, false>(a, nt, cw, st);
    else
        e = always ? launch_resident_typed<uint64_t, true, false>(a, nt, cw, st)
            : rare ? launch_resident_typed<uint64_t, false, true>(a, nt, cw, st)
                   : launch_resident_typed<uint64_t, false, false>(a, nt, cw, st);
    if (e == cudaSuccess) {
        s->resident_epoch += 4 * n;
        s->count_launch();
    }
    return e;
}

} // namespace ea

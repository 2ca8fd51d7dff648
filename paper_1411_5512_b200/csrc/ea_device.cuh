// ea_device.cuh -- device-side building blocks shared by the kernels of libea_b200.so.
//
// Everything here implements the WRITTEN stream contract of DESIGN.md section 2 (C-xx) for the
// paper's update (Manssen & Hartmann, arXiv:1411.5512; section III).  It shares no
// code with oracle/ (the CPU checker is written independently from the same text).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ea {

// ---------------------------------------------------------------------------------------------
// HBM layout.  Sites are split by colour c = (x+y+z)&1 and compacted along x:
//   compact index i = xh + Lh*(y + L*z),  xh = x>>1,  Lh = L/2,  x = 2*xh + (c ^ ((y+z)&1)).
//   spins  : uint64 [2][Nh]           (Nh = N/2)
//   bonds  : BondT  [2][3][Nh]        forward bond (d, site) stored at the site's (colour, compact index);
//            BondT = uint64 for 64 independent samples, uint32 for 32 disorders x 2 replicas
//            (hi half == lo half by PAPER.md:33, so only the low half is stored and read).
// A half-sweep of colour c reads spins[c], spins[1-c], all six bond planes once and writes spins[c].
// ---------------------------------------------------------------------------------------------
struct Lattice {
    int L, Lh;       // side, side/2
    int log2Lh;      // >= 0 if Lh is a power of two, else -1
    int log2L;       // >= 0 if L is a power of two, else -1
    unsigned Nh;     // L^3 / 2
};

// Philox4x32-10 (Salmon et al., SC'11), reading C-A6: multipliers 0xD2511F53 (on c0) and
// 0xCD9E8D57 (on c2), Weyl increments 0x9E3779B9 / 0xBB67AE85 added to the key after each round.
constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;

// Stream tags, 4th counter word (C-A6).
enum : uint32_t { TAG_PARITY0 = 0, TAG_PARITY1 = 1, TAG_INIT_SPINS = 2, TAG_BONDS = 3 };

__device__ __forceinline__ void mulhilo(uint32_t a, uint32_t b, uint32_t &hi, uint32_t &lo)
{
    unsigned long long p = (unsigned long long)a * (unsigned long long)b; // one IMAD.WIDE.U32
    hi = (uint32_t)(p >> 32);
    lo = (uint32_t)p;
}

// The full block function (all four outputs); used by the setup kernels and the self-test.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0, l0, h1, l1;
        mulhilo(PHILOX_M0, c0, h0, l0);
        mulhilo(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The update stream of one half-sweep (C-A6, C-A7): the same-colour sites of an x-row, j = x >> 1 = compact index
// xh, pair up (xh even, xh + 1) and share ONE block per sweep: counter (site index of the pair's first site,
// t lo, t hi, parity), key = seed; the first site takes out[0] (samples 0..31) and out[1] (samples 32..63), the
// second out[2] and out[3].  Only c0 varies inside a launch, so everything that depends on (t, parity, seed)
// alone is folded once per launch into SweepRng (rounds 1-2 collapse to two multiplies).
// The result is bit-identical to philox4x32_10(first site, t lo, t hi, parity; seed).
struct SweepRng {
    uint32_t x2;     // tag ^ k1[0]
    uint32_t x0;     // lo(M1*t_hi) ^ k0[1]
    uint32_t y2;     // hi(M0*U0) ^ k1[1],  U0 = hi(M1*t_hi) ^ t_lo ^ k0[0]
    uint32_t z2;     // lo(M0*U0) ^ k1[2]
    uint32_t k0[10]; // round keys (only [2..9] used)
    uint32_t k1[10]; // round keys (only [3..9] used)
};

__host__ __device__ inline SweepRng make_sweep_rng(uint64_t seed, uint64_t t, uint32_t tag)
{
    SweepRng g;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        g.k0[r] = k0 + (uint32_t)r * PHILOX_W0;
        g.k1[r] = k1 + (uint32_t)r * PHILOX_W1;
    }
    uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
    uint64_t p1 = (uint64_t)PHILOX_M1 * t_hi;
    uint32_t U0 = (uint32_t)(p1 >> 32) ^ t_lo ^ g.k0[0];
    uint32_t U1 = (uint32_t)p1;
    uint64_t q0 = (uint64_t)PHILOX_M0 * U0;
    g.x2 = tag ^ g.k1[0];
    g.x0 = U1 ^ g.k0[1];
    g.y2 = (uint32_t)(q0 >> 32) ^ g.k1[1];
    g.z2 = (uint32_t)q0 ^ g.k1[2];
    return g;
}

// Same folding when the round keys are already in place (RESIDENT: keys arrive as kernel parameters).
__host__ __device__ inline void sweep_rng_set_time(SweepRng &g, uint64_t t, uint32_t tag)
{
    uint32_t t_lo = (uint32_t)t, t_hi = (uint32_t)(t >> 32);
    uint64_t p1 = (uint64_t)PHILOX_M1 * t_hi;
    uint32_t U0 = (uint32_t)(p1 >> 32) ^ t_lo ^ g.k0[0];
    uint32_t U1 = (uint32_t)p1;
    uint64_t q0 = (uint64_t)PHILOX_M0 * U0;
    g.x2 = tag ^ g.k1[0];
    g.x0 = U1 ^ g.k0[1];
    g.y2 = (uint32_t)(q0 >> 32) ^ g.k1[1];
    g.z2 = (uint32_t)q0 ^ g.k1[2];
}

__device__ __forceinline__ uint4 sweep_random4(const SweepRng &g, uint32_t first_site)
{
    uint32_t h, l, h0, l0, h1, l1;
    // round 1: (site, t_lo, t_hi, tag) -> (U0, U1, n2, n3)
    mulhilo(PHILOX_M0, first_site, h, l);
    uint32_t n2 = h ^ g.x2, n3 = l;
    // round 2: (U0, U1, n2, n3) -> (m0, m1, m2, V3)
    mulhilo(PHILOX_M1, n2, h, l);
    uint32_t c0 = h ^ g.x0, c1 = l, c2 = n3 ^ g.y2;
    // round 3: c3 = V3 is launch-uniform
    mulhilo(PHILOX_M0, c0, h0, l0);
    mulhilo(PHILOX_M1, c2, h1, l1);
    c0 = h1 ^ c1 ^ g.k0[2];
    c1 = l1;
    c2 = h0 ^ g.z2;
    uint32_t c3 = l0;
    // rounds 4..10
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        mulhilo(PHILOX_M0, c0, h0, l0);
        mulhilo(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ g.k0[r];
        c1 = l1;
        c2 = h0 ^ c3 ^ g.k1[r];
        c3 = l0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// the two numbers of ONE site: `second` = xh & 1 selects the half of its pair's block (scalar kernel, self-test)
__device__ __forceinline__ void sweep_random(const SweepRng &g, uint32_t first_site, unsigned second, uint32_t &r_lo,
                                             uint32_t &r_hi)
{
    const uint4 o = sweep_random4(g, first_site);
    r_lo = second ? o.z : o.x;
    r_hi = second ? o.w : o.y;
}

// Acceptance thresholds of Eq. 9 (C-A4) prepared for 32-bit compares:
// accept at n_u = k  <=>  r < thr[k]  with thr[k] in [0, 2^32];  thr == 2^32 ("always", T = inf)
// does not fit a 32-bit compare, so it is carried as an all-ones mask OR-ed into the result.
struct Thresholds {
    uint32_t thr[3];    // min(thr[k], 2^32 - 1)
    uint32_t always[3]; // 0xffffffff if thr[k] == 2^32 else 0
    // heat-bath variant (reading C-HB; not the paper's dynamics): P(flip | n_u) = 1 / (1 + exp((12 - 4 n_u) / T)),
    // n_u = 0..6, increasing in n_u; same clamping
    uint32_t hb[7];
    uint32_t hb_always[7];
};

// one LOP3 with truth table LUT over (a, b, c) = (0xF0, 0xCC, 0xAA); plain asm (not volatile): free to schedule, but the
// compiler cannot take the expression apart into two-input operations
template <int LUT> __device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return d;
}
constexpr int LUT_XOR3 = 0x96, LUT_MAJ = 0xE8, LUT_MAJ_NA = 0x8E; // a ^ b ^ c;  maj(a, b, c);  maj(~a, b, c)

__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c) { return a ^ b ^ c; }
__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c) { return (a & b) | (c & (a | b)); }

// One 32-sample half of one Metropolis trial (Eq. 9; "boolean logic at the bit level").
// u1..u6: unsatisfied-bond words j ^ sigma_i ^ sigma_nbr (C-A2, C-A3).  Two full adders give
// a = u1+u2+u3 = sa + 2 ka and b = u4+u5+u6 = sb + 2 kb, n_u = a + b.  With t = sa | sb:
//   [n_u >= 3] = maj(ka, kb, t),  [n_u >= 2] = ka | kb | (sa & sb),  [n_u >= 1] = ka | kb | t.
// The thresholds are nested (thr[0] <= thr[1] <= thr[2]), so
//   f = [n_u >= 3] | [r < thr[2]] [n_u >= 2] | [r < thr[1]] [n_u >= 1] | [r < thr[0]]
// and each rare term is one or two predicated LOP3 behind an ISETP (no masks are materialised).
// ALWAYS: some thr[k] == 2^32 (T = inf), which a 32-bit compare cannot express -- OR-ed in as masks.
struct HalfCount { uint32_t sa, ka, sb, kb; };

__device__ __forceinline__ HalfCount count_half(uint32_t u1, uint32_t u2, uint32_t u3, uint32_t u4, uint32_t u5, uint32_t u6)
{
    HalfCount h;
    h.sa = xor3(u1, u2, u3); h.ka = maj3(u1, u2, u3);
    h.sb = xor3(u4, u5, u6); h.kb = maj3(u4, u5, u6);
    return h;
}

__device__ __forceinline__ HalfCount count_half_lop3(uint32_t u1, uint32_t u2, uint32_t u3, uint32_t u4, uint32_t u5, uint32_t u6)
{
    HalfCount h;
    h.sa = lop3<LUT_XOR3>(u1, u2, u3); h.ka = lop3<LUT_MAJ>(u1, u2, u3);
    h.sb = lop3<LUT_XOR3>(u4, u5, u6); h.kb = lop3<LUT_MAJ>(u4, u5, u6);
    return h;
}

// the energy-raising levels of one half, given that r < thr[2] is possible
__device__ __forceinline__ uint32_t raise_half(uint32_t f, const HalfCount &h, uint32_t r, const Thresholds &th)
{
    const uint32_t t = h.sa | h.sb;
    if (r < th.thr[2]) f = h.ka | h.kb | (h.sa & h.sb);
    if (r < th.thr[1]) f = h.ka | h.kb | t;
    if (r < th.thr[0]) f = 0xffffffffu;
    return f;
}

template <bool ALWAYS>
__device__ __forceinline__ uint32_t flip_half(uint32_t u1, uint32_t u2, uint32_t u3, uint32_t u4, uint32_t u5,
                                              uint32_t u6, uint32_t r, const Thresholds &th)
{
    const HalfCount h = count_half(u1, u2, u3, u4, u5, u6);
    const uint32_t t = h.sa | h.sb;
    uint32_t f = raise_half(maj3(h.ka, h.kb, t), h, r, th);
    if (ALWAYS) f |= (th.always[2] & (h.ka | h.kb | (h.sa & h.sb))) | (th.always[1] & (h.ka | h.kb | t)) | th.always[0];
    return f;
}

// Heat bath (C-HB): flip iff r < hb[n_u].  hb is increasing in n_u, so with k* the smallest k with r < hb[k] the spin flips
// iff n_u >= k*.  In terms of a_d = j_d ^ n_d and their number n_a (n_u = n_a for s = 0, 6 - n_a for s = 1) the NEW spin is
// [n_a >= k*] for s = 0 and [n_a >= 7 - k*] for s = 1; with the two full adders (sa, ka), (sb, kb) of the a_d and
// M(x; a, b) = maj(x, a, b),  A = M(~s; ka, kb), A' = M(s; ka, kb), B = M(~s; sa, sb), B' = M(s; sa, sb):
//   k* = 0: ~s   1: M(~s; A, B)   2: M(~s; A, B')   3: maj(ka, kb, B)   4: maj(ka, kb, B')   5: M(s; A', B)   6: M(s; A', B')   7: s
// -- a chain of seven predicated assignments from k = 6 down to 0 (the last one taken is k*).  hb[k] == 2^32 (T = 0,
// Delta E < 0: certain whatever r) cannot be expressed by the 32-bit compare and rides on hb_always[k].
__device__ __forceinline__ uint32_t new_spin_half_heatbath(uint32_t s, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t a4, uint32_t a5,
                                                           uint32_t a6, uint32_t r, const Thresholds &th)
{
    const HalfCount h = count_half_lop3(a1, a2, a3, a4, a5, a6);
    const uint32_t A = lop3<LUT_MAJ_NA>(s, h.ka, h.kb), A2 = lop3<LUT_MAJ>(s, h.ka, h.kb);
    const uint32_t B = lop3<LUT_MAJ_NA>(s, h.sa, h.sb), B2 = lop3<LUT_MAJ>(s, h.sa, h.sb);
    uint32_t n = s;
    if (r < th.hb[6] || th.hb_always[6]) n = lop3<LUT_MAJ>(s, A2, B2);
    if (r < th.hb[5] || th.hb_always[5]) n = lop3<LUT_MAJ>(s, A2, B);
    if (r < th.hb[4] || th.hb_always[4]) n = lop3<LUT_MAJ>(h.ka, h.kb, B2);
    if (r < th.hb[3] || th.hb_always[3]) n = lop3<LUT_MAJ>(h.ka, h.kb, B);
    if (r < th.hb[2] || th.hb_always[2]) n = lop3<LUT_MAJ_NA>(s, A, B2);
    if (r < th.hb[1] || th.hb_always[1]) n = lop3<LUT_MAJ_NA>(s, A, B);
    if (r < th.hb[0] || th.hb_always[0]) n = ~s;
    return n;
}

// 64-bit word <-> halves
__device__ __forceinline__ uint32_t lo32(uint64_t w) { return (uint32_t)w; }
__device__ __forceinline__ uint32_t hi32(uint64_t w) { return (uint32_t)(w >> 32); }
__device__ __forceinline__ uint64_t mk64(uint32_t lo, uint32_t hi) { return (uint64_t)lo | ((uint64_t)hi << 32); }

// Bond word -> the two 32-sample halves the update logic needs.
__device__ __forceinline__ uint32_t bond_lo(uint64_t j) { return (uint32_t)j; }
__device__ __forceinline__ uint32_t bond_hi(uint64_t j) { return (uint32_t)(j >> 32); }
__device__ __forceinline__ uint32_t bond_lo(uint32_t j) { return j; }
__device__ __forceinline__ uint32_t bond_hi(uint32_t j) { return j; } // replica (b) sees the same bonds

// One whole Metropolis trial of a 64-sample word: returns the new spin word.  (n_d, j_d), d = 1..6: the six
// neighbour words with the bond word that couples each to this site, in any order (n_u is a count).
// RARE (low temperature, thr[2] << 2^32): the three energy-raising levels sit behind ONE warp-level branch per
// word, taken only if some lane drew r < thr[2] in either half (T = 0.8: 0.7 % per draw, 35 % per warp and word),
// instead of six compares and eight predicated LOP3 on the alu pipe that binds these kernels.  Same result.
template <typename BondT, bool ALWAYS, bool RARE = false, bool HB = false>
__device__ __forceinline__ uint64_t metropolis_word(uint64_t s, uint64_t n1, uint64_t n2, uint64_t n3, uint64_t n4,
                                                    uint64_t n5, uint64_t n6, BondT j1, BondT j2, BondT j3, BondT j4,
                                                    BondT j5, BondT j6, uint32_t r_lo, uint32_t r_hi,
                                                    const Thresholds &th)
{
    const uint32_t sl = lo32(s), sh = hi32(s);
    if (HB) {
        const uint32_t nl = new_spin_half_heatbath(sl, bond_lo(j1) ^ lo32(n1), bond_lo(j2) ^ lo32(n2), bond_lo(j3) ^ lo32(n3),
                                                   bond_lo(j4) ^ lo32(n4), bond_lo(j5) ^ lo32(n5), bond_lo(j6) ^ lo32(n6), r_lo, th);
        const uint32_t nh = new_spin_half_heatbath(sh, bond_hi(j1) ^ hi32(n1), bond_hi(j2) ^ hi32(n2), bond_hi(j3) ^ hi32(n3),
                                                   bond_hi(j4) ^ hi32(n4), bond_hi(j5) ^ hi32(n5), bond_hi(j6) ^ hi32(n6), r_hi, th);
        return mk64(nl, nh);
    }
    if (RARE && !ALWAYS) {
        // In terms of a_d = j_d ^ n_d (J S_nbr = -1 seen from an up spin) and n_a = their number, n_u = n_a for s = 0 and
        // 6 - n_a for s = 1, so the NEW spin is  s' = [n_a >= 3 - l] (s = 0),  [n_a >= 4 + l] (s = 1),  l = 0..3 the number
        // of thresholds above r.  With the two full adders n_a = sa + sb + 2 (ka + kb) and M(x; a, b) = maj(x, a, b)
        // (x = 1: a | b, x = 0: a & b):   l = 0:  s' = maj(ka, kb, M(~s; sa, sb))      -- 12 LOP3 per half, no s ^ f
        //   l = 1:  s' = M(~s; M(~s; ka, kb), M(s; sa, sb))     l = 2:  s' = M(~s; M(~s; ka, kb), M(~s; sa, sb))     l = 3:  ~s
        const HalfCount hl = count_half_lop3(bond_lo(j1) ^ lo32(n1), bond_lo(j2) ^ lo32(n2), bond_lo(j3) ^ lo32(n3),
                                             bond_lo(j4) ^ lo32(n4), bond_lo(j5) ^ lo32(n5), bond_lo(j6) ^ lo32(n6));
        const HalfCount hh = count_half_lop3(bond_hi(j1) ^ hi32(n1), bond_hi(j2) ^ hi32(n2), bond_hi(j3) ^ hi32(n3),
                                             bond_hi(j4) ^ hi32(n4), bond_hi(j5) ^ hi32(n5), bond_hi(j6) ^ hi32(n6));
        const uint32_t tl = lop3<LUT_MAJ_NA>(sl, hl.sa, hl.sb), th_ = lop3<LUT_MAJ_NA>(sh, hh.sa, hh.sb);
        uint32_t nl = lop3<LUT_MAJ>(hl.ka, hl.kb, tl), nh = lop3<LUT_MAJ>(hh.ka, hh.kb, th_);
        if (min(r_lo, r_hi) < th.thr[2]) {
            if (r_lo < th.thr[2]) {
                const uint32_t u = r_lo < th.thr[1] ? tl : lop3<LUT_MAJ>(sl, hl.sa, hl.sb);
                nl = lop3<LUT_MAJ_NA>(sl, lop3<LUT_MAJ_NA>(sl, hl.ka, hl.kb), u);
                if (r_lo < th.thr[0]) nl = ~sl;
            }
            if (r_hi < th.thr[2]) {
                const uint32_t u = r_hi < th.thr[1] ? th_ : lop3<LUT_MAJ>(sh, hh.sa, hh.sb);
                nh = lop3<LUT_MAJ_NA>(sh, lop3<LUT_MAJ_NA>(sh, hh.ka, hh.kb), u);
                if (r_hi < th.thr[0]) nh = ~sh;
            }
        }
        return mk64(nl, nh);
    }
    if (!ALWAYS) { // every temperature: the same new-spin formulation with the three levels predicated (no branch)
        const HalfCount hl = count_half_lop3(bond_lo(j1) ^ lo32(n1), bond_lo(j2) ^ lo32(n2), bond_lo(j3) ^ lo32(n3),
                                             bond_lo(j4) ^ lo32(n4), bond_lo(j5) ^ lo32(n5), bond_lo(j6) ^ lo32(n6));
        const HalfCount hh = count_half_lop3(bond_hi(j1) ^ hi32(n1), bond_hi(j2) ^ hi32(n2), bond_hi(j3) ^ hi32(n3),
                                             bond_hi(j4) ^ hi32(n4), bond_hi(j5) ^ hi32(n5), bond_hi(j6) ^ hi32(n6));
        const uint32_t tl = lop3<LUT_MAJ_NA>(sl, hl.sa, hl.sb), th_ = lop3<LUT_MAJ_NA>(sh, hh.sa, hh.sb);
        uint32_t nl = lop3<LUT_MAJ>(hl.ka, hl.kb, tl), nh = lop3<LUT_MAJ>(hh.ka, hh.kb, th_);
        const uint32_t xl = lop3<LUT_MAJ_NA>(sl, hl.ka, hl.kb), xh = lop3<LUT_MAJ_NA>(sh, hh.ka, hh.kb);
        if (r_lo < th.thr[2]) nl = lop3<LUT_MAJ_NA>(sl, xl, lop3<LUT_MAJ>(sl, hl.sa, hl.sb));
        if (r_lo < th.thr[1]) nl = lop3<LUT_MAJ_NA>(sl, xl, tl);
        if (r_lo < th.thr[0]) nl = ~sl;
        if (r_hi < th.thr[2]) nh = lop3<LUT_MAJ_NA>(sh, xh, lop3<LUT_MAJ>(sh, hh.sa, hh.sb));
        if (r_hi < th.thr[1]) nh = lop3<LUT_MAJ_NA>(sh, xh, th_);
        if (r_hi < th.thr[0]) nh = ~sh;
        return mk64(nl, nh);
    }
    const uint32_t fl = flip_half<ALWAYS>(bond_lo(j1) ^ sl ^ lo32(n1), bond_lo(j2) ^ sl ^ lo32(n2),
                                          bond_lo(j3) ^ sl ^ lo32(n3), bond_lo(j4) ^ sl ^ lo32(n4),
                                          bond_lo(j5) ^ sl ^ lo32(n5), bond_lo(j6) ^ sl ^ lo32(n6), r_lo, th);
    const uint32_t fh = flip_half<ALWAYS>(bond_hi(j1) ^ sh ^ hi32(n1), bond_hi(j2) ^ sh ^ hi32(n2),
                                          bond_hi(j3) ^ sh ^ hi32(n3), bond_hi(j4) ^ sh ^ hi32(n4),
                                          bond_hi(j5) ^ sh ^ hi32(n5), bond_hi(j6) ^ sh ^ hi32(n6), r_hi, th);
    return mk64(sl ^ fl, sh ^ fh);
}

// ---------------------------------------------------------------------------------------------
// 32x32 bit-matrix transpose across a warp (observables: per-sample popcounts).
// In : lane i holds w_i, bit j of w_i = sample j at site i.   Out: lane j holds bit i = sample j at site i.
// Five butterfly stages; stage s swaps bit s of the lane index with bit s of the bit index.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t warp_transpose32(uint32_t w, unsigned lane)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        // keep-mask: bit positions whose bit-s equals the lane's bit-s stay; the others come from the partner
        const uint32_t lowmask = (s == 16) ? 0x0000ffffu : (s == 8) ? 0x00ff00ffu : (s == 4) ? 0x0f0f0f0fu
                                 : (s == 2)                                                 ? 0x33333333u
                                                                                            : 0x55555555u;
        uint32_t p = __shfl_xor_sync(0xffffffffu, w, s);
        if (lane & s)
            w = (w & ~lowmask) | ((p >> s) & lowmask);
        else
            w = (w & lowmask) | ((p << s) & ~lowmask);
    }
    return w;
}

} // namespace ea

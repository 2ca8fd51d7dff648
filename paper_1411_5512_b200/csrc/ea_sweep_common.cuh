// ea_sweep_common.cuh -- device helpers shared by the half-sweep kernels (ea_sweep.cu: one launch per colour;
// ea_sweep_resident.cu: persistent, lattice resident in shared memory).  All variants run the same update
// (Eq. 9) through metropolis_word() and are bit-identical.
#pragma once
#include "ea_device.cuh"

namespace ea {

template <typename T> struct Pair;
template <> struct Pair<uint64_t> { typedef ulonglong2 type; };
template <> struct Pair<uint32_t> { typedef uint2 type; };

template <typename BondT>
__device__ __forceinline__ void ld_pair(const BondT *p, BondT &a, BondT &b)
{
    typename Pair<BondT>::type v = __ldg((const typename Pair<BondT>::type *)p);
    a = v.x;
    b = v.y;
}

template <typename BondT>
__device__ __forceinline__ typename Pair<BondT>::type ldg_pair(const BondT *p)
{
    return __ldg((const typename Pair<BondT>::type *)p);
}

__device__ __forceinline__ uint64_t shfl64(uint64_t v, int src)
{
    uint32_t lo = __shfl_sync(0xffffffffu, lo32(v), src), hi = __shfl_sync(0xffffffffu, hi32(v), src);
    return mk64(lo, hi);
}
__device__ __forceinline__ uint32_t shfl_bond(uint32_t v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ uint64_t shfl_bond(uint64_t v, int src) { return shfl64(v, src); }

// The update of the lane's two words given their four random numbers r = (word 0 lo/hi half, word 1 lo/hi half).
template <int S, typename BondT, bool ALWAYS, bool RARE = false, bool HB = false>
__device__ __forceinline__ ulonglong2 update_pair_r(const ulonglong2 own, const ulonglong2 P0, const ulonglong2 Pm,
                                                    const ulonglong2 Pp, const ulonglong2 Zm, const ulonglong2 Zp,
                                                    const typename Pair<BondT>::type jx,
                                                    const typename Pair<BondT>::type jy,
                                                    const typename Pair<BondT>::type jz,
                                                    const typename Pair<BondT>::type bx,
                                                    const typename Pair<BondT>::type by,
                                                    const typename Pair<BondT>::type bz, const uint4 r,
                                                    const Thresholds &th, const int lane_m, const int lane_p)
{
    ulonglong2 out;
    if (S == 0) { // own x = 4k, 4k+2; other colour at 4k+1 (P0.x), 4k+3 (P0.y), 4k-1 (left lane's P0.y)
        const uint64_t ex = shfl64(P0.y, lane_m);
        const BondT jex = shfl_bond((BondT)bx.y, lane_m);
        out.x = metropolis_word<BondT, ALWAYS, RARE, HB>(own.x, P0.x, ex, Pp.x, Pm.x, Zp.x, Zm.x, (BondT)jx.x, jex, (BondT)jy.x,
                                               (BondT)by.x, (BondT)jz.x, (BondT)bz.x, r.x, r.y, th);
        out.y = metropolis_word<BondT, ALWAYS, RARE, HB>(own.y, P0.y, P0.x, Pp.y, Pm.y, Zp.y, Zm.y, (BondT)jx.y, (BondT)bx.x,
                                               (BondT)jy.y, (BondT)by.y, (BondT)jz.y, (BondT)bz.y, r.z, r.w, th);
    } else {      // own x = 4k+1, 4k+3; other colour at 4k (P0.x), 4k+2 (P0.y), 4k+4 (right lane's P0.x)
        const uint64_t ex = shfl64(P0.x, lane_p);
        out.x = metropolis_word<BondT, ALWAYS, RARE, HB>(own.x, P0.y, P0.x, Pp.x, Pm.x, Zp.x, Zm.x, (BondT)jx.x, (BondT)bx.x,
                                               (BondT)jy.x, (BondT)by.x, (BondT)jz.x, (BondT)bz.x, r.x, r.y, th);
        out.y = metropolis_word<BondT, ALWAYS, RARE, HB>(own.y, ex, P0.y, Pp.y, Pm.y, Zp.y, Zm.y, (BondT)jx.y, (BondT)bx.y,
                                               (BondT)jy.y, (BondT)by.y, (BondT)jz.y, (BondT)bz.y, r.z, r.w, th);
    }
    return out;
}

template <int S, typename BondT, bool ALWAYS, bool RARE = false, bool HB = false>
__device__ __forceinline__ ulonglong2 update_pair(const ulonglong2 own, const ulonglong2 P0, const ulonglong2 Pm,
                                                  const ulonglong2 Pp, const ulonglong2 Zm, const ulonglong2 Zp,
                                                  const typename Pair<BondT>::type jx,
                                                  const typename Pair<BondT>::type jy,
                                                  const typename Pair<BondT>::type jz,
                                                  const typename Pair<BondT>::type bx,
                                                  const typename Pair<BondT>::type by,
                                                  const typename Pair<BondT>::type bz, const uint32_t site0,
                                                  const SweepRng &g, const Thresholds &th, const int lane_m,
                                                  const int lane_p)
{
    const uint4 r = sweep_random4(g, site0); // the lane's two words are one pair (xh = 2k, 2k + 1): one block
    return update_pair_r<S, BondT, ALWAYS, RARE, HB>(own, P0, Pm, Pp, Zm, Zp, jx, jy, jz, bx, by, bz, r, th, lane_m, lane_p);
}

} // namespace ea

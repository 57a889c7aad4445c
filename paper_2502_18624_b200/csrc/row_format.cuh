// How one thread's slice of a colour row (32 same-colour sites) sits in memory and in
// registers, for the nibble-arithmetic kernels (update.cu, observe.cu).
//
// 4-bit models (ISING, BLUME_CAPEL): one 128-bit vector, nibble j of 32-bit half q = site 8q + j.
// ISING_MODEL_BLUME_CAPEL_2BIT (NEXT-3, "2 bits per spin"): one 64-bit vector, site j
// of a 32-bit half at bits 2j..2j+1.  It is expanded to nibbles in registers by an even/odd split
//     E = w & 0x33333333 (nibble j = site 2j),   O = (w >> 2) & 0x33333333 (nibble j = site 2j + 1)
// and the register words are ordered (x, y, z, w) = (E_lo, O_lo, E_hi, O_hi).  The in-row neighbour
// of an even site is an odd site and vice versa, so one of the two side words is a plain copy.
#pragma once

#include "ising_internal.cuh"

template <int MODEL> struct RowFmt {
    static constexpr bool kTwoBit = MODEL == ISING_MODEL_BLUME_CAPEL_2BIT;
    static constexpr int kVecBytes = kTwoBit ? 8 : 16;      // bytes per thread per row
    static constexpr int kHalves = kVecBytes / 4;           // 32-bit halves per vector
};

template <int MODEL>
__device__ __forceinline__ uint4 load_row(const char *ptr)
{
    if (RowFmt<MODEL>::kTwoBit) {
        const uint2 v = *reinterpret_cast<const uint2 *>(ptr);
        return make_uint4(v.x & 0x33333333u, (v.x >> 2) & 0x33333333u, v.y & 0x33333333u, (v.y >> 2) & 0x33333333u);
    }
    return *reinterpret_cast<const uint4 *>(ptr);
}

template <int MODEL>
__device__ __forceinline__ void store_row(char *ptr, const uint4 &o)
{
    if (RowFmt<MODEL>::kTwoBit) *reinterpret_cast<uint2 *>(ptr) = make_uint2(o.x | (o.y << 2), o.z | (o.w << 2));
    else *reinterpret_cast<uint4 *>(ptr) = o;
}

// side word: for row parity p = (y + colour) & 1 the in-row neighbour that is not at the same
// compact index k is k-1 (p = 0) or k+1 (p = 1)  [SURVEY.md Sec. 8 conventions].  `edge` is the
// raw 32-bit half next to the vector (see edge_half) that supplies the one site across its border.
template <int MODEL, int P>
__device__ __forceinline__ void side_words(const uint4 &sm, uint32_t edge, uint32_t sd[4])
{
    if (RowFmt<MODEL>::kTwoBit) {
        if (P == 0) {  // site 2j - 1 = O nibble j - 1 for the even sites, site 2j = E nibble j for the odd ones
            sd[0] = __funnelshift_l(edge >> 2, sm.y, 4);       // top nibble of (edge >> 2) = site 15 of the previous half
            sd[1] = sm.x;
            sd[2] = __funnelshift_l(sm.y, sm.w, 4);
            sd[3] = sm.z;
        } else {       // site 2j + 1 = O nibble j for the even sites, site 2j + 2 = E nibble j + 1 for the odd ones
            sd[0] = sm.y;
            sd[1] = __funnelshift_r(sm.x, sm.z, 4);
            sd[2] = sm.w;
            sd[3] = __funnelshift_r(sm.z, edge & 3u, 4);       // site 0 of the next half
        }
    } else if (P == 0) {  // neighbour k-1: shift nibbles up, carry in the top nibble of the previous half
        sd[0] = __funnelshift_l(edge, sm.x, 4);
        sd[1] = __funnelshift_l(sm.x, sm.y, 4);
        sd[2] = __funnelshift_l(sm.y, sm.z, 4);
        sd[3] = __funnelshift_l(sm.z, sm.w, 4);
    } else {              // neighbour k+1: shift nibbles down, carry in the bottom nibble of the next half
        sd[0] = __funnelshift_r(sm.x, sm.y, 4);
        sd[1] = __funnelshift_r(sm.y, sm.z, 4);
        sd[2] = __funnelshift_r(sm.z, sm.w, 4);
        sd[3] = __funnelshift_r(sm.w, edge, 4);
    }
}

// index (in 32-bit halves, within the row) of the half that supplies the site across the border
template <int MODEL, int P>
__device__ __forceinline__ int edge_half(int col, int cols)
{
    constexpr int H = RowFmt<MODEL>::kHalves;
    if (P == 0) return (col == 0) ? cols * H - 1 : H * col - 1;
    return (col == cols - 1) ? 0 : H * col + H;
}

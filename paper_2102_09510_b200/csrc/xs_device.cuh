// xs_device.cuh -- device helpers shared by the kernels: LOP3 truth tables, the Boolean QG
// update (a-4..a-7), Philox4x32-10 (a-6), vector shared/global accessors.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "xs_internal.h"

namespace xs {

// ------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return d;
}
// LUT index = a*4 + b*2 + c
constexpr int LUT_XOR3 = 0x96;
constexpr int LUT_MAJ = 0xE8;
constexpr int LUT_MAJ_NOTC = 0xD4;   // maj(a, b, ~c)
constexpr int LUT_SEL = 0xCA;        // a ? b : c
constexpr int LUT_NZ = 0x7E;         // (a^c)|(b^c): not all equal

// Philox4x32-10 (Salmon et al., SC'11).  ctr = (c0,c1,c2,c3), key = (k0,k1).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t o[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0);
        const uint32_t l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2);
        const uint32_t l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0;
        c2 = h0 ^ c3 ^ k1;
        c1 = l1;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

// Same with the 10 round keys precomputed (the key is fixed per instance: keeps the key
// schedule's 20 additions out of every call).
__device__ __forceinline__ void philox_key_schedule(uint32_t k0, uint32_t k1, uint32_t (&ks)[10][2])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        ks[r][0] = k0 + (uint32_t)r * 0x9E3779B9u;
        ks[r][1] = k1 + (uint32_t)r * 0xBB67AE85u;
    }
}
__device__ __forceinline__ void philox4x32_10_ks(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 const uint32_t (&ks)[10][2], uint32_t o[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0);
        const uint32_t l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2);
        const uint32_t l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ ks[r][0];
        c2 = h0 ^ c3 ^ ks[r][1];
        c1 = l1;
        c3 = l0;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

// One QG update of 32 clones.  a*/b* partner words, j* coupling masks, x own word, R noise mask.
__device__ __forceinline__ uint32_t qg_update(uint32_t a0, uint32_t b0, uint32_t j0, uint32_t a1,
                                              uint32_t b1, uint32_t j1, uint32_t a2, uint32_t b2,
                                              uint32_t j2, uint32_t x, uint32_t R)
{
    const uint32_t w0 = lop3<LUT_XOR3>(a0, b0, j0);
    const uint32_t w1 = lop3<LUT_XOR3>(a1, b1, j1);
    const uint32_t w2 = lop3<LUT_XOR3>(a2, b2, j2);
    const uint32_t M = lop3<LUT_MAJ>(w0, w1, w2);
    const uint32_t P = lop3<LUT_XOR3>(w0, w1, w2);
    const uint32_t f = lop3<LUT_MAJ_NOTC>(M, P, x);
    return lop3<LUT_SEL>(R, f, M);
}
// General flip table (PAPER.md: w_k = probability of flipping a spin that enters k
// unsatisfied interactions; L69: w0 = w1^3 gives detailed balance).  Rk = all-ones iff the
// word's number is below the threshold of w_k.  k = 2 (M^x) + (P^x) selects the mask:
//   flip = (M^x) ? ((P^x) ? R3 : R2) : ((P^x) ? R1 : R0)
__device__ __forceinline__ uint32_t table_update(uint32_t a0, uint32_t b0, uint32_t j0, uint32_t a1,
                                                 uint32_t b1, uint32_t j1, uint32_t a2, uint32_t b2,
                                                 uint32_t j2, uint32_t x, uint32_t R0, uint32_t R1,
                                                 uint32_t R2, uint32_t R3)
{
    const uint32_t w0 = lop3<LUT_XOR3>(a0, b0, j0);
    const uint32_t w1 = lop3<LUT_XOR3>(a1, b1, j1);
    const uint32_t w2 = lop3<LUT_XOR3>(a2, b2, j2);
    const uint32_t Mu = lop3<LUT_MAJ>(w0, w1, w2) ^ x;
    const uint32_t Pu = lop3<LUT_XOR3>(w0, w1, w2) ^ x;
    const uint32_t lo = lop3<LUT_SEL>(Pu, R1, R0);
    const uint32_t hi = lop3<LUT_SEL>(Pu, R3, R2);
    return x ^ lop3<LUT_SEL>(Mu, hi, lo);
}

// Bits set where the spin has k != 0 unsatisfied clauses.
__device__ __forceinline__ uint32_t qg_nonzero_k(uint32_t a0, uint32_t b0, uint32_t j0, uint32_t a1,
                                                 uint32_t b1, uint32_t j1, uint32_t a2, uint32_t b2,
                                                 uint32_t j2, uint32_t x)
{
    const uint32_t w0 = lop3<LUT_XOR3>(a0, b0, j0);
    const uint32_t w1 = lop3<LUT_XOR3>(a1, b1, j1);
    const uint32_t w2 = lop3<LUT_XOR3>(a2, b2, j2);
    const uint32_t M = lop3<LUT_MAJ>(w0, w1, w2);
    const uint32_t P = lop3<LUT_XOR3>(w0, w1, w2);
    return lop3<LUT_NZ>(M, P, x);
}

// CW uint64 words handled by one lane, as 2*CW uint32.
template <int CW> struct Vec;
template <> struct Vec<1> { uint2 v; };
template <> struct Vec<2> { uint4 v; };

template <int CW> __device__ __forceinline__ void vload(const void* p, uint32_t (&o)[2 * CW]);
template <> __device__ __forceinline__ void vload<1>(const void* p, uint32_t (&o)[2])
{
    const uint2 t = *reinterpret_cast<const uint2*>(p);
    o[0] = t.x; o[1] = t.y;
}
template <> __device__ __forceinline__ void vload<2>(const void* p, uint32_t (&o)[4])
{
    const uint4 t = *reinterpret_cast<const uint4*>(p);
    o[0] = t.x; o[1] = t.y; o[2] = t.z; o[3] = t.w;
}
template <int CW> __device__ __forceinline__ void vstore(void* p, const uint32_t (&o)[2 * CW]);
template <> __device__ __forceinline__ void vstore<1>(void* p, const uint32_t (&o)[2])
{
    *reinterpret_cast<uint2*>(p) = make_uint2(o[0], o[1]);
}
template <> __device__ __forceinline__ void vstore<2>(void* p, const uint32_t (&o)[4])
{
    *reinterpret_cast<uint4*>(p) = make_uint4(o[0], o[1], o[2], o[3]);
}


// per-clone Bernoulli(m / 128) mask of 32 clones.  r[k] holds bit k of the
// clones' 7-bit numbers U (bit-sliced); returns the mask of clones with U < m by a most significant
// bit first comparison against the constant m (m >= 128: all clones).
__device__ __forceinline__ uint32_t clone_noise_mask(const uint32_t (&r)[7], uint32_t m)
{
    if (m >= 128u) return ~0u;
    uint32_t lt = 0u, eq = ~0u;
#pragma unroll
    for (int k = 6; k >= 0; --k) {
        if ((m >> k) & 1u) { lt |= eq & ~r[k]; eq &= r[k]; }
        else               { eq &= ~r[k]; }
    }
    return lt;
}

}  // namespace xs

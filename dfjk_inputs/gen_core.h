/*
 * gen_core.h -- counter-based random numbers and the synthetic-B element formula.
 *
 * INPUT GENERATION ONLY.  This module holds none of the DF-JK arithmetic: it
 * neither forms densities nor contracts anything.  It serves both the oracle's
 * tests and the CUDA path's tests/bench with the SAME bytes; neither of those
 * two includes the other.
 *
 * Recipe (BASELINE.json configs):
 *   x_mu      = sort( U(0,10) )                         basis-function "centres"
 *   a_P       = U(0.05,1) * exp(-P/naux)                P = 0..naux-1
 *   z_P,pair ~ N(0,1), one draw per PACKED index (mu >= nu)  => symmetric by construction
 *   Bp[P][mu(mu+1)/2+nu] = a_P * exp(-(x_mu-x_nu)^2/4) * (1 + 0.1 z_P,pair)
 *
 * Random numbers: every value is a pure function of (seed, stream, index), so any
 * element can be produced anywhere, in any order, on host or device.
 */
#ifndef DFJK_GEN_CORE_H
#define DFJK_GEN_CORE_H
#include <stdint.h>
#include <math.h>

#ifdef __CUDACC__
#define GEN_HD __host__ __device__ __forceinline__
#else
#define GEN_HD static inline
#endif

/* splitmix64 finaliser */
GEN_HD uint64_t gen_fmix(uint64_t z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

GEN_HD uint64_t gen_key(uint64_t seed, uint64_t stream)
{
    return gen_fmix(gen_fmix(seed + 0x9E3779B97F4A7C15ULL) ^
                    gen_fmix((stream + 1) * 0xD1B54A32D192ED03ULL));
}

/* integer stage: the part that is bit-identical on host and device */
GEN_HD uint64_t gen_bits(uint64_t key, uint64_t index)
{
    return gen_fmix(key + (index + 1) * 0x9E3779B97F4A7C15ULL);
}

/* U in (0,1), 53 bits */
GEN_HD double gen_u01(uint64_t key, uint64_t index)
{
    return ((double)(gen_bits(key, index) >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* N(0,1): Box-Muller from counters 2*index, 2*index+1 */
GEN_HD double gen_normal(uint64_t key, uint64_t index)
{
    const double u1 = gen_u01(key, 2 * index);
    const double u2 = gen_u01(key, 2 * index + 1);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

/* streams */
#define GEN_STREAM_X 0u
#define GEN_STREAM_A 1u
#define GEN_STREAM_Z 2u
#define GEN_STREAM_C 10u   /* + 16*call + set */
#define GEN_STREAM_ROT 1000u /* + 16*call + set */

/* locality factor g(mu,nu) = exp(-(x_mu-x_nu)^2/4) */
GEN_HD double gen_locality(double xm, double xn)
{
    const double dx = xm - xn;
    return exp(-0.25 * dx * dx);
}

/* one element of packed B */
GEN_HD double gen_b_elem(uint64_t zkey, double aP, double g, uint64_t flat_index)
{
    return aP * g * (1.0 + 0.1 * gen_normal(zkey, flat_index));
}

#endif

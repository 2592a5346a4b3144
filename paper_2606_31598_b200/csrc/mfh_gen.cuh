// mfh_gen.cuh -- device generator: Philox4x32-10 words -> Box-Muller normals -> GUE entries.
//
// One Philox call per unordered pair {i,j}: key = seed, ctr = (min(i,j), max(i,j), stream, 0)
// (BASELINE.json configs[0]; partition invariance P:68-70: global indices only).
// Used by the fused generate-and-apply kernels, the cache fill and the debug exports, so the
// cached and the procedural path apply bit-identical matrices.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mfh {

// Round keys k + r*W are seed-only constants: computed once on the host, passed by value in the
// kernel parameter block (constant bank), so each round's xor takes them as immediate operands.
struct PhiloxKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

inline PhiloxKeys make_philox_keys(uint64_t seed)
{
    PhiloxKeys K;
    uint32_t a = (uint32_t)(seed & 0xffffffffu), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        K.k0[r] = a;
        K.k1[r] = b;
        a += 0x9E3779B9u;
        b += 0xBB67AE85u;
    }
    return K;
}

// Full 4-word output.  In the fused kernels only x0,x1 are consumed and the compiler removes the
// dead half of the last two rounds.
__device__ __forceinline__ void philox4x32_10(const PhiloxKeys& K, uint32_t c0, uint32_t c1,
                                              uint32_t c2, uint32_t c3, uint32_t& x0, uint32_t& x1,
                                              uint32_t& x2, uint32_t& x3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;   // IMAD.WIDE.U32
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];    // LOP3
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    x0 = c0; x1 = c1; x2 = c2; x3 = c3;
}

// Words (x0,x1) of the matrix stream for an ordered pair lo <= hi.
__device__ __forceinline__ void pair_words(const PhiloxKeys& K, uint32_t lo, uint32_t hi,
                                           uint32_t& x0, uint32_t& x1)
{
    uint32_t x2, x3;
    philox4x32_10(K, lo, hi, 0u, 0u, x0, x1, x2, x3);
}

// ---- Box-Muller normals scaled by s:  (s*g1, s*g2),  g1 + i g2 = sqrt(-2 ln u1) e^{2 pi i u2},
//      u = (x + 1/2) 2^-32  (readings R2, R3). --------------------------------------

template <typename T> struct Gen;

template <> struct Gen<double> {
    __device__ __forceinline__ static void normals(uint32_t x0, uint32_t x1, double s, double& a,
                                                   double& b)
    {
        // 2^52 + x as a double by bit pattern, then one exact FMA: (x + 1/2) 2^-32.
        const double d0 = __hiloint2double(0x43300000, (int)x0);
        const double d1 = __hiloint2double(0x43300000, (int)x1);
        const double u1 = fma(d0, 0x1p-32, -(0x1p52 - 0.5) * 0x1p-32);
        const double two_u2 = fma(d1, 0x1p-31, -(0x1p52 - 0.5) * 0x1p-31);
        const double r = s * sqrt(-2.0 * log(u1));
        double sn, cs;
        sincospi(two_u2, &sn, &cs);
        a = r * cs;
        b = r * sn;
    }
};

template <> struct Gen<float> {
    __device__ __forceinline__ static void normals(uint32_t x0, uint32_t x1, float s, float& a,
                                                   float& b)
    {
        // u1 rounded to float (may round to 1 -> r = 0; error <= 6e-8, R6).
        const float u1 = fmaf((float)x0, 0x1p-32f, 0x1p-33f);
        // angle as a signed turn fraction in [-1/2, 1/2): same angle mod 1, full float precision
        const float two_u2 = fmaf((float)(int32_t)x1, 0x1p-31f, 0x1p-32f);
        const float r = s * sqrtf(-2.0f * logf(u1));
        float sn, cs;
        sincospif(two_u2, &sn, &cs);
        a = r * cs;
        b = r * sn;
    }
};

// Scales of the entry rule: off-diagonal 1/sqrt(2D), diagonal 1/sqrt(D).
template <typename T> struct Scales {
    T off;
    T diag;
};

// General entry H_ij for any (i,j): conjugate below the diagonal, real on it.
template <typename T>
__device__ __forceinline__ void entry_any(const PhiloxKeys& K, const Scales<T>& S, uint32_t i,
                                          uint32_t j, T& hr, T& hi)
{
    uint32_t x0, x1;
    pair_words(K, min(i, j), max(i, j), x0, x1);
    T a, b;
    Gen<T>::normals(x0, x1, (i == j) ? S.diag : S.off, a, b);
    hr = a;
    hi = (i < j) ? b : ((i > j) ? -b : T(0));
}

// Entry for a pair known to satisfy i < j (strictly upper triangle).
template <typename T>
__device__ __forceinline__ void entry_upper(const PhiloxKeys& K, const Scales<T>& S, uint32_t i,
                                            uint32_t j, T& hr, T& hi)
{
    uint32_t x0, x1;
    pair_words(K, i, j, x0, x1);
    Gen<T>::normals(x0, x1, S.off, hr, hi);
}

}  // namespace mfh

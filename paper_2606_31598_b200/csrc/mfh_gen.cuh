// mfh_gen.cuh -- device generator: Philox4x32-10 words -> Box-Muller normals -> GUE entries.
//
// One Philox call per unordered pair {i,j}: key = seed, ctr = (min(i,j), max(i,j), stream, 0)
// (BASELINE.json configs[0]; partition invariance P:68-70: global indices only).
// Used by the fused generate-and-apply kernels, the cache fill and the debug exports, so the
// cached and the procedural path apply bit-identical matrices.
//
// The Box-Muller transcendentals are this file's own: the
// fused c128 kernel is bound by issue slots and the FP64 pipe, and libdevice's 1-ulp log / sqrt /
// sincospi cost ~210 instructions per entry; the table-driven forms below cost ~50 and keep the
// absolute error of an entry below 1e-13 of its scale (tolerance of phi: 1e-11 relative L2).
#pragma once
#include <cstddef>
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

// 32x32 -> 64 multiply by a Philox constant.  Written as PTX: from the C expression
// (uint64_t)M * x nvcc emits the IMAD.WIDE plus an extra integer add per product; the wide multiply
// issues at a quarter of the FP32 rate on sm_100 and is the scarcest pipe of the generator.
__device__ __forceinline__ void mul_m0(uint32_t x, uint32_t& lo, uint32_t& hi)
{
    uint64_t p;
    asm("mul.wide.u32 %0, %1, 0xD2511F53;" : "=l"(p) : "r"(x));
    lo = (uint32_t)p;
    hi = (uint32_t)(p >> 32);
}
__device__ __forceinline__ void mul_m1(uint32_t x, uint32_t& lo, uint32_t& hi)
{
    uint64_t p;
    asm("mul.wide.u32 %0, %1, 0xCD9E8D57;" : "=l"(p) : "r"(x));
    lo = (uint32_t)p;
    hi = (uint32_t)(p >> 32);
}

// Full 4-word output (debug export, H0 diagonal).
__device__ __forceinline__ void philox4x32_10(const PhiloxKeys& K, uint32_t c0, uint32_t c1,
                                              uint32_t c2, uint32_t c3, uint32_t& x0, uint32_t& x1,
                                              uint32_t& x2, uint32_t& x3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t lo0, hi0, lo1, hi1;
        mul_m0(c0, lo0, hi0);
        mul_m1(c2, lo1, hi1);
        const uint32_t n0 = hi1 ^ c1 ^ K.k0[r];    // LOP3
        const uint32_t n2 = hi0 ^ c3 ^ K.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    x0 = c0; x1 = c1; x2 = c2; x3 = c3;
}

// Words (x0,x1) of the matrix stream for an ordered pair lo <= hi: counter (lo, hi, 0, 0).  The zero
// counter words remove one multiply from the first round, the unused words x2,x3 one from the last:
// 18 wide multiplies and 18 three-input xors per call.
__device__ __forceinline__ void pair_words(const PhiloxKeys& K, uint32_t lo, uint32_t hi,
                                           uint32_t& x0, uint32_t& x1)
{
    uint32_t lo0, hi0, lo1, hi1;
    mul_m0(lo, lo0, hi0);                           // round 0: c2 = c3 = 0
    uint32_t c0 = hi ^ K.k0[0], c1 = 0u, c2 = hi0 ^ K.k1[0], c3 = lo0;
#pragma unroll
    for (int r = 1; r < 9; ++r) {
        mul_m0(c0, lo0, hi0);
        mul_m1(c2, lo1, hi1);
        const uint32_t n0 = hi1 ^ c1 ^ K.k0[r];
        const uint32_t n2 = hi0 ^ c3 ^ K.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    mul_m1(c2, lo1, hi1);                           // round 9: only x0, x1 are consumed
    x0 = hi1 ^ c1 ^ K.k0[9];
    x1 = lo1;
}

// ---- Box-Muller normals scaled by s = 1/sqrt(2D):  (s g1, s g2),
//      g1 + i g2 = sqrt(-2 ln u1) e^{2 pi i u2},  u = (x + 1/2) 2^-32   (R2, R3). ------
//
// complex128.  With d = x0 + 1/2 = 2^e m (m in [1,2)), c the centre of m's bin among 256 and
// r = m/c - 1 (|r| <= 2^-9):
//     L = s^2 (-2 ln u1) = K2 [(32 - e) ln 2 - ln c] - K2 log1p(r),      K2 = 2 s^2 = 1/D,
// a 256-entry table of (1/c, -K2 ln c), a 33-entry table of K2 (32-e) ln 2 and a degree-4
// polynomial for log1p (remainder r^5/5 <= 6e-15).  sqrt(L) = L y (1 + e + 3/2 e^2), y = rsqrt.approx(L)
// (2^-21), e = 1/2 - 1/2 L y^2: third-order correct (1e-19 relative).  The angle 2 pi u2 is split into a
// 1024-entry table of (cos A, sin A) at the bin centres and a residual |b| <= pi/1024 (b = (x1 mod 2^22) ang - 2^21 ang:
// sin b = b - b^3/6 (2e-15), cos b = 1 - b^2/2 + b^4/24 (1e-18), combined by angle addition.
constexpr int GEN_LOG_BITS = 8;
constexpr int GEN_SC_BITS = 10;

struct GenTabD {                         // built on the host by make_gen_table(), copied to shared memory
    double2 tsc[1 << GEN_SC_BITS];       // (cos A, sin A),  A = 2 pi (idx 2^22 + 2^21 + 1/2) 2^-32
    double2 tlog[1 << GEN_LOG_BITS];     // (1/c, -K2 ln c)
    double elog[34];                     // K2 (32 - e) ln 2 for e = -1..31  (index e + 1)
};
// The shared-memory copy every generating kernel stages (stage_gen_table): a FILE-SCOPE __shared__ object, so that
// its address is a compile-time constant inside each kernel.
__shared__ __align__(16) GenTabD g_gen_tab_d;

struct GenConstD {                       // kernel-parameter constants (constant bank operands)
    double c1, c2, c3, c4;               // -K2 log1p(r) = r (c1 + r (c2 + r (c3 + r c4)))
    double ang;                          // 2 pi 2^-32
    double ang_off;                      // -2^21 ang: centres the residual angle, folded into one FMA
};

struct GenHostD {
    GenTabD tab;
    GenConstD gc;
};

void make_gen_table(int64_t D, GenHostD& out);   // mfh_plan.cu (host)

template <typename T> struct Gen;

template <> struct Gen<double> {
    using Tab = GenTabD;
    using Const = GenConstD;
    static constexpr int TAB_BYTES = (int)sizeof(GenTabD);

    __device__ __forceinline__ static void normals(const GenTabD*, const GenConstD& gc,
                                                   uint32_t x0, uint32_t x1, double& a, double& b)
    {
        // radius: d = x0 + 1/2 exactly (2^52 + x0 by bit pattern, minus 2^52 - 1/2)
        const double d = __hiloint2double(0x43300000, (int)x0) - 0x1.fffffffffffffp51;
        const uint32_t hi = (uint32_t)__double2hiint(d);
        uint32_t mh;                                                     // mantissa with exponent 0: one LOP3
        asm("lop3.b32 %0, %1, 0x000fffff, 0x3ff00000, 0xEA;" : "=r"(mh) : "r"(hi));
        const double m = __hiloint2double((int)mh, __double2loint(d));
        // byte offsets of the look-ups; the table is a file-scope __shared__ object, so its address is a compile-time
        // constant that folds into the immediate of each LDS (no integer add for the base)
        const char* tb = reinterpret_cast<const char*>(&g_gen_tab_d);
        const double2 tl = *reinterpret_cast<const double2*>(tb + offsetof(GenTabD, tlog) + ((hi >> (20 - GEN_LOG_BITS - 4)) & (((1u << GEN_LOG_BITS) - 1u) << 4)));
        const double el = *reinterpret_cast<const double*>(tb + ((int)offsetof(GenTabD, elog) - 1022 * 8) + ((hi >> 17) & 0x3ff8u));
        const double r = fma(m, tl.x, -1.0);
        double p = fma(r, gc.c4, gc.c3);
        p = fma(r, p, gc.c2);
        p = fma(r, p, gc.c1);
        const double L = fma(r, p, tl.y + el);
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(L));
        // sqrt(L) = sq (1 + e/2 + 3/8 e^2 + O(e^3)) with sq = L y, e = 1 - L y^2 (|e| <= 2^-20): the second-order
        // term removes the -3/2 delta^2 bias a single Newton step would leave in every entry (1.9e-13, which a
        // Chebyshev propagation over 151 applies would add up)
        const double sq = L * y;
        const double e = fma(-sq, y, 1.0);
        const double rad = fma(sq, e * fma(e, 0.375, 0.5), sq);
        // angle: residual of x1 inside its bin, centred by the constant term of one FMA (exact: 2^21 ang is ang scaled
        // by a power of two)
        const double2 cs = *reinterpret_cast<const double2*>(tb + offsetof(GenTabD, tsc) + ((x1 >> (32 - GEN_SC_BITS - 4)) & (((1u << GEN_SC_BITS) - 1u) << 4)));
        const double bb = fma((double)(int)(x1 & ((1u << (32 - GEN_SC_BITS)) - 1u)), gc.ang, gc.ang_off);
        const double b2 = bb * bb;
        const double sb = fma(b2 * (-1.0 / 6.0), bb, bb);
        const double q = fma(b2, 1.0 / 24.0, -0.5) * b2;
        const double rc = rad * cs.x, rs = rad * cs.y;
        a = fma(-rs, sb, fma(rc, q, rc));
        b = fma(rc, sb, fma(rs, q, rs));
    }
};

// complex64: SFU forms (lg2 / sqrt / sin / cos .approx, absolute error <= 5e-7 per normal;
// tolerance of phi: 1e-4).  u1 is rounded to float (may round to 1 -> radius 0; R6);
// the angle is taken as a signed turn fraction in [-1/2, 1/2) so the SFU argument stays in [-pi, pi).
struct GenTabF {
    float unused;
};
struct GenConstF {
    float neg_k2_ln2;   // -K2 ln 2:  L = K2 (-ln u1) = neg_k2_ln2 * log2(u1)
};

template <> struct Gen<float> {
    using Tab = GenTabF;
    using Const = GenConstF;
    static constexpr int TAB_BYTES = 0;

    __device__ __forceinline__ static void normals(const GenTabF*, const GenConstF& gc, uint32_t x0,
                                                   uint32_t x1, float& a, float& b)
    {
        // .ftz SFU forms: no denormal fix-up branches (u1 >= 2^-33, L >= 0, |turn| <= 1/2)
        const float u1 = fmaf((float)x0, 0x1p-32f, 0x1p-33f);
        float lg, rad, cs, sn;
        asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(u1));
        const float L = gc.neg_k2_ln2 * lg;
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(rad) : "f"(L));
        const float ang = fmaf((float)(int32_t)x1, 0x1.921fb6p-30f, 0x1.921fb6p-31f);   // 2 pi (x1 + 1/2) 2^-32
        asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cs) : "f"(ang));
        asm("sin.approx.ftz.f32 %0, %1;" : "=f"(sn) : "f"(ang));
        a = rad * cs;
        b = rad * sn;
    }
};

// Analytic source (Eq. 9; R22): H_ij = -t e^{+i phi} / (j - i)^alpha for i < j, its
// conjugate for i > j, H_ii = W cos(2 pi beta i + delta).  cos/sin of phi and 2 pi beta are prepared on the host.
struct AnalyticArgs {
    double t, alpha, cphi, sphi, W, beta2pi, delta;
};
enum { SRC_SEEDED = 0, SRC_ANALYTIC = 1 };   // template parameter of the kernels that generate entries

template <typename T> struct GenArgs {   // what a kernel needs to call the generator
    PhiloxKeys K;
    typename Gen<T>::Const gc;
    const typename Gen<T>::Tab* tab_global;   // device copy of the table (nullptr for float)
    AnalyticArgs an;                          // SRC_ANALYTIC only
};

// Entry of the analytic source, evaluated in double (pow, cos) and rounded to T.
template <typename T>
__device__ __forceinline__ void analytic_entry(const AnalyticArgs& A, uint32_t i, uint32_t j, T& hr, T& hi)
{
    if (i == j) {
        hr = (T)(A.W * cos(fma(A.beta2pi, (double)i, A.delta)));
        hi = T(0);
        return;
    }
    const double d = (double)(i < j ? j - i : i - j);
    const double a = -A.t * pow(d, -A.alpha);
    hr = (T)(a * A.cphi);
    hi = (T)(i < j ? a * A.sphi : -(a * A.sphi));
}

// Copy the generator table to shared memory (all threads of the CTA; caller synchronises).
template <typename T>
__device__ __forceinline__ const typename Gen<T>::Tab* stage_gen_table(const GenArgs<T>& G)
{
    if constexpr (Gen<T>::TAB_BYTES > 0) {
        const uint4* src = reinterpret_cast<const uint4*>(G.tab_global);
        uint4* dst = reinterpret_cast<uint4*>(&g_gen_tab_d);
        for (int t = threadIdx.x; t < Gen<T>::TAB_BYTES / 16; t += blockDim.x) dst[t] = src[t];
        return &g_gen_tab_d;
    } else {
        return nullptr;
    }
}

// General entry H_ij for any (i,j): conjugate below the diagonal, real and scaled by 1/sqrt(D)
// (= sqrt(2) s) on it.
template <typename T, int SRC = SRC_SEEDED>
__device__ __forceinline__ void entry_any(const GenArgs<T>& G, const typename Gen<T>::Tab* tab, uint32_t i,
                                          uint32_t j, T& hr, T& hi)
{
    if constexpr (SRC == SRC_ANALYTIC) {
        analytic_entry<T>(G.an, i, j, hr, hi);
        return;
    }
    uint32_t x0, x1;
    pair_words(G.K, min(i, j), max(i, j), x0, x1);
    T a, b;
    Gen<T>::normals(tab, G.gc, x0, x1, a, b);
    hr = (i == j) ? a * T(1.4142135623730951) : a;
    hi = (i < j) ? b : ((i > j) ? -b : T(0));
}

// Entry for a pair known to satisfy i < j (strictly upper triangle).
template <typename T, int SRC = SRC_SEEDED>
__device__ __forceinline__ void entry_upper(const GenArgs<T>& G, const typename Gen<T>::Tab* tab, uint32_t i,
                                            uint32_t j, T& hr, T& hi)
{
    if constexpr (SRC == SRC_ANALYTIC) {
        analytic_entry<T>(G.an, i, j, hr, hi);
        return;
    }
    uint32_t x0, x1;
    pair_words(G.K, i, j, x0, x1);
    Gen<T>::normals(tab, G.gc, x0, x1, hr, hi);
}

// Entry for a pair known to satisfy i > j: conjugate of the (j,i) entry.
template <typename T, int SRC = SRC_SEEDED>
__device__ __forceinline__ void entry_lower(const GenArgs<T>& G, const typename Gen<T>::Tab* tab, uint32_t i,
                                            uint32_t j, T& hr, T& hi)
{
    if constexpr (SRC == SRC_ANALYTIC) {
        analytic_entry<T>(G.an, i, j, hr, hi);
        return;
    }
    uint32_t x0, x1;
    pair_words(G.K, j, i, x0, x1);
    T b;
    Gen<T>::normals(tab, G.gc, x0, x1, hr, b);
    hi = -b;
}

}  // namespace mfh

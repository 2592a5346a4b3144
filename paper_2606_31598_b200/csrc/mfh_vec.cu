// mfh_vec.cu -- O(D) vector kernels: the fixed-order reduction of partial sums with the
// H0 + lambda V epilogue (BASELINE.json configs[2]) and the Chebyshev recurrence updates
// (Eq. 41-44).  All are HBM-trivial next to the O(D^2) apply.
#include <algorithm>
#include <cstdint>
#include "mfh_internal.cuh"

namespace mfh {

struct LamArr {
    double v[MFH_MAX_K];
};

// phi[i][v] = h0_i psi[i][v] + lambda_v * sum_{valid slots s} work[s][i][v]; the valid slots of a
// block row come as a compact ascending list.  A CTA handles 64 consecutive elements with 4 thread
// groups: group g adds the g-th quarter of the list (four loads in flight), the quarters are
// combined in the order 0..3 through shared memory: a fixed summation order that does not depend
// on CTA scheduling (no atomics).  Needs B*k to be a multiple of 64 so that the 64 elements of a
// CTA share one block row; the launcher falls back to 1 group x 256 elements otherwise.
constexpr int RED_E = 64, RED_G = 4;

template <typename T, int G>
__global__ void __launch_bounds__(256) reduce_kernel(int64_t D, int32_t B, int32_t k, int32_t n_slots,
                                                     const int32_t* __restrict__ slot_list,
                                                     const typename Cplx<T>::type* __restrict__ work,
                                                     const T* __restrict__ h0,
                                                     const typename Cplx<T>::type* __restrict__ psi,
                                                     typename Cplx<T>::type* __restrict__ phi, LamArr lam)
{
    using CT = typename Cplx<T>::type;
    constexpr int EPB = 256 / G;                       // elements per CTA
    __shared__ double part[G][EPB][2];
    const int64_t total = D * k;
    const int ex = threadIdx.x % EPB, g = threadIdx.x / EPB;
    for (int64_t e0 = (int64_t)blockIdx.x * EPB; e0 < total; e0 += (int64_t)gridDim.x * EPB) {
        const int64_t e = e0 + ex;
        const bool live = e < total;
        const int64_t i = live ? e / k : 0;
        const int32_t* list = slot_list + (size_t)(i / B) * (n_slots + 1);   // [count, slots...]
        const int head = list[0];                                             // count | SLOT_* flags
        const int cnt = head & SLOT_COUNT_MASK;
        const int chunk = (cnt + G - 1) / G;
        int t = g * chunk;
        const int t_end = live ? min(cnt, t + chunk) : 0;
        double sr = 0.0, si = 0.0;
        for (; t + 4 <= t_end; t += 4) {
            const CT x0 = work[(size_t)list[1 + t] * total + e];
            const CT x1 = work[(size_t)list[2 + t] * total + e];
            const CT x2 = work[(size_t)list[3 + t] * total + e];
            const CT x3 = work[(size_t)list[4 + t] * total + e];
            sr += (double)x0.x; si += (double)x0.y;
            sr += (double)x1.x; si += (double)x1.y;
            sr += (double)x2.x; si += (double)x2.y;
            sr += (double)x3.x; si += (double)x3.y;
        }
        for (; t < t_end; ++t) {
            const CT x = work[(size_t)list[1 + t] * total + e];
            sr += (double)x.x;
            si += (double)x.y;
        }
        if (G > 1) {
            part[g][ex][0] = sr;
            part[g][ex][1] = si;
            __syncthreads();
            if (g == 0)
#pragma unroll
                for (int gg = 1; gg < G; ++gg) {
                    sr += part[gg][ex][0];
                    si += part[gg][ex][1];
                }
        }
        if (g == 0 && live && !(head & SLOT_SKIP_ROW)) {
            const int v = (int)(e - i * k);
            double outr = lam.v[v] * sr, outi = lam.v[v] * si;
            if (h0 && !(head & SLOT_NO_H0)) {
                const CT p = psi[e];
                const double d = (double)h0[i];
                outr = fma(d, (double)p.x, outr);
                outi = fma(d, (double)p.y, outi);
            }
            CT o;
            o.x = (T)outr;
            o.y = (T)outi;
            phi[e] = o;
        }
        if (G > 1) __syncthreads();
    }
}

// complex64 with many slots (the k-vector plans with column-side slots, C3: 32 .. 280 per block row): the same fixed
// summation order, two neighbouring elements per thread (one 16-byte load per slot, eight in flight).  One CTA per 64
// element pairs, the LAST block rows first: the slot count grows with the block row, and the hardware scheduler
// balances a heaviest-first list of CTAs.
__global__ void __launch_bounds__(256) reduce2_kernel_c64(int64_t D, int32_t B, int32_t k, int32_t n_slots,
                                                          const int32_t* __restrict__ slot_list, const float2* __restrict__ work,
                                                          const float* __restrict__ h0, const float2* __restrict__ psi,
                                                          float2* __restrict__ phi, LamArr lam)
{
    constexpr int G = RED_G, EPB = 256 / G;              // element PAIRS per CTA
    __shared__ double part[G][EPB][4];
    const int64_t total = D * k;                         // k even: a pair never crosses a row
    const int ex = threadIdx.x % EPB, g = threadIdx.x / EPB;
    const int64_t e = 2 * (((int64_t)gridDim.x - 1 - blockIdx.x) * EPB + ex);
    const bool live = e < total;
    const int64_t i = live ? e / k : 0;
    const int32_t* list = slot_list + (size_t)(i / B) * (n_slots + 1);
    const int head = list[0];
    const int cnt = head & SLOT_COUNT_MASK;
    const int chunk = (cnt + G - 1) / G;
    int t = g * chunk;
    const int t_end = live ? min(cnt, t + chunk) : 0;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    for (; t + 8 <= t_end; t += 8) {
        float4 x[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) x[u] = *reinterpret_cast<const float4*>(work + (size_t)list[1 + t + u] * total + e);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            s0 += (double)x[u].x; s1 += (double)x[u].y; s2 += (double)x[u].z; s3 += (double)x[u].w;
        }
    }
    for (; t < t_end; ++t) {
        const float4 x = *reinterpret_cast<const float4*>(work + (size_t)list[1 + t] * total + e);
        s0 += (double)x.x; s1 += (double)x.y; s2 += (double)x.z; s3 += (double)x.w;
    }
    part[g][ex][0] = s0; part[g][ex][1] = s1; part[g][ex][2] = s2; part[g][ex][3] = s3;
    __syncthreads();
    if (g != 0 || !live || (head & SLOT_SKIP_ROW)) return;
#pragma unroll
    for (int gg = 1; gg < G; ++gg) {
        s0 += part[gg][ex][0]; s1 += part[gg][ex][1]; s2 += part[gg][ex][2]; s3 += part[gg][ex][3];
    }
    const int v = (int)(e - i * k);
    double o0 = lam.v[v] * s0, o1 = lam.v[v] * s1, o2 = lam.v[v + 1] * s2, o3 = lam.v[v + 1] * s3;
    if (h0 && !(head & SLOT_NO_H0)) {
        const float4 p = *reinterpret_cast<const float4*>(psi + e);
        const double d = (double)h0[i];
        o0 = fma(d, (double)p.x, o0); o1 = fma(d, (double)p.y, o1);
        o2 = fma(d, (double)p.z, o2); o3 = fma(d, (double)p.w, o3);
    }
    *reinterpret_cast<float4*>(phi + e) = make_float4((float)o0, (float)o1, (float)o2, (float)o3);
}

template <typename T, int G>
static int launch_reduce_t(mfh_handle h, const void* psi, void* phi, const LamArr& lam, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    const Plan& p = h->plan;
    const int64_t total = h->D * p.k;
    const int epb = 256 / G;
    const int blocks = (int)std::min<int64_t>((total + epb - 1) / epb, (int64_t)h->sm_count * 8);
    reduce_kernel<T, G><<<blocks, 256, 0, st>>>(h->D, p.B, p.k, std::max(p.n_slots, 1), h->d_slot_list,
                                                 (const CT*)h->d_work, (const T*)h->d_h0, (const CT*)psi, (CT*)phi, lam);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_reduce(mfh_handle h, const void* psi, void* phi, const double* lambdas, cudaStream_t st)
{
    const Plan& p = h->plan;
    LamArr lam;
    for (int v = 0; v < MFH_MAX_K; ++v) lam.v[v] = (v < p.k) ? (lambdas ? lambdas[v] : h->lambda) : 0.0;
    const bool split = ((int64_t)p.B * p.k) % RED_E == 0 && p.n_slots >= 16;
    if (h->dtype == MFH_C64 && split && p.k % 2 == 0 && p.n_slots >= 64 && ((uintptr_t)psi % 16 == 0) && ((uintptr_t)phi % 16 == 0)) {
        const int64_t pairs = h->D * p.k / 2;
        const int epb = 256 / RED_G;
        reduce2_kernel_c64<<<(unsigned)((pairs + epb - 1) / epb), 256, 0, st>>>(h->D, p.B, p.k, std::max(p.n_slots, 1), h->d_slot_list,
                                                                                (const float2*)h->d_work, (const float*)h->d_h0,
                                                                                (const float2*)psi, (float2*)phi, lam);
        MFH_CUDA_CHECK(cudaGetLastError());
        return MFH_OK;
    }
    if (h->dtype == MFH_C128)
        return split ? launch_reduce_t<double, RED_G>(h, psi, phi, lam, st) : launch_reduce_t<double, 1>(h, psi, phi, lam, st);
    return split ? launch_reduce_t<float, RED_G>(h, psi, phi, lam, st) : launch_reduce_t<float, 1>(h, psi, phi, lam, st);
}

// ---- Chebyshev -------------------------------------------------------------------------------
// first:  q0 = psi, acc = J_0 q0                                            (Eq. 41)
// step:   next = first ? (Hq - c q)/R : 2 (Hq - c q)/R - prev               (Eq. 42, 43)
//         dst = next;  acc += coef * next      (coef = 2 (-i)^l J_l(a), complex)
// final:  out = e^{-ict} acc
template <typename T>
__global__ void cheb_first_kernel(int64_t D, const typename Cplx<T>::type* __restrict__ psi,
                                  typename Cplx<T>::type* __restrict__ q0,
                                  typename Cplx<T>::type* __restrict__ acc, double j0)
{
    using CT = typename Cplx<T>::type;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < D;
         i += (int64_t)gridDim.x * blockDim.x) {
        const CT p = psi[i];
        q0[i] = p;
        CT a;
        a.x = (T)(j0 * (double)p.x);
        a.y = (T)(j0 * (double)p.y);
        acc[i] = a;
    }
}

template <typename T>
__global__ void cheb_step_kernel(int64_t D, const typename Cplx<T>::type* __restrict__ hq,
                                 const typename Cplx<T>::type* __restrict__ q,
                                 typename Cplx<T>::type* prev_dst, typename Cplx<T>::type* __restrict__ acc,
                                 double c, double inv_r, int first, double cr, double ci)
{
    using CT = typename Cplx<T>::type;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < D;
         i += (int64_t)gridDim.x * blockDim.x) {
        const CT hv = hq[i], qv = q[i];
        double nr = ((double)hv.x - c * (double)qv.x) * inv_r;
        double ni = ((double)hv.y - c * (double)qv.y) * inv_r;
        if (!first) {
            const CT pv = prev_dst[i];
            nr = 2.0 * nr - (double)pv.x;
            ni = 2.0 * ni - (double)pv.y;
        }
        CT nx;
        nx.x = (T)nr;
        nx.y = (T)ni;
        prev_dst[i] = nx;
        CT a = acc[i];
        a.x = (T)((double)a.x + cr * nr - ci * ni);
        a.y = (T)((double)a.y + cr * ni + ci * nr);
        acc[i] = a;
    }
}

template <typename T>
__global__ void cheb_final_kernel(int64_t D, const typename Cplx<T>::type* __restrict__ acc,
                                  typename Cplx<T>::type* __restrict__ out, double pr, double pi)
{
    using CT = typename Cplx<T>::type;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < D;
         i += (int64_t)gridDim.x * blockDim.x) {
        const CT a = acc[i];
        CT o;
        o.x = (T)(pr * (double)a.x - pi * (double)a.y);
        o.y = (T)(pr * (double)a.y + pi * (double)a.x);
        out[i] = o;
    }
}

static int vec_blocks(mfh_handle h) { return (int)std::min<int64_t>((h->D * h->plan.k + 255) / 256, (int64_t)h->sm_count * 8); }

int launch_cheb_first(mfh_handle h, const void* psi, void* q0, void* acc, double j0, cudaStream_t st)
{
    if (h->dtype == MFH_C128)
        cheb_first_kernel<double><<<vec_blocks(h), 256, 0, st>>>(h->D * h->plan.k, (const double2*)psi, (double2*)q0, (double2*)acc, j0);
    else
        cheb_first_kernel<float><<<vec_blocks(h), 256, 0, st>>>(h->D * h->plan.k, (const float2*)psi, (float2*)q0, (float2*)acc, j0);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_cheb_step(mfh_handle h, const void* hq, const void* q, void* prev_dst, void* acc, double c,
                     double inv_r, int first, double coef_re, double coef_im, cudaStream_t st)
{
    if (h->dtype == MFH_C128)
        cheb_step_kernel<double><<<vec_blocks(h), 256, 0, st>>>(h->D * h->plan.k, (const double2*)hq, (const double2*)q, (double2*)prev_dst,
                                                                 (double2*)acc, c, inv_r, first, coef_re, coef_im);
    else
        cheb_step_kernel<float><<<vec_blocks(h), 256, 0, st>>>(h->D * h->plan.k, (const float2*)hq, (const float2*)q, (float2*)prev_dst,
                                                                (float2*)acc, c, inv_r, first, coef_re, coef_im);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_cheb_final(mfh_handle h, const void* acc, void* out, double ph_re, double ph_im, cudaStream_t st)
{
    if (h->dtype == MFH_C128)
        cheb_final_kernel<double><<<vec_blocks(h), 256, 0, st>>>(h->D * h->plan.k, (const double2*)acc, (double2*)out, ph_re, ph_im);
    else
        cheb_final_kernel<float><<<vec_blocks(h), 256, 0, st>>>(h->D * h->plan.k, (const float2*)acc, (float2*)out, ph_re, ph_im);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// ---- Lanczos ("matrix-free Lanczos iterations estimate spectral bounds") ----------------
// All scalars stay on the device (alpha[], beta[] arrays), so the m steps run without a host
// synchronisation; reductions are two-stage (per-CTA partial, then one CTA adds the partials in
// index order): deterministic.
constexpr int LZ_BLOCKS = 296, LZ_THREADS = 256;

template <typename T>
__device__ __forceinline__ void block_sum2(double& a, double& b)
{
    __shared__ double sa[LZ_THREADS / 32], sb[LZ_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (w == 0) {
        a = lane < LZ_THREADS / 32 ? sa[lane] : 0.0;
        b = lane < LZ_THREADS / 32 ? sb[lane] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, o);
            b += __shfl_xor_sync(0xffffffffu, b, o);
        }
    }
}

// partial[2b], partial[2b+1] = sum over CTA b's elements of conj(x) y  (x == y gives the squared norm)
template <typename T>
__global__ void __launch_bounds__(LZ_THREADS) lz_dot_kernel(int64_t D, const typename Cplx<T>::type* __restrict__ x,
                                                            const typename Cplx<T>::type* __restrict__ y,
                                                            double* __restrict__ partial)
{
    double re = 0.0, im = 0.0;
    for (int64_t i = blockIdx.x * (int64_t)LZ_THREADS + threadIdx.x; i < D; i += (int64_t)gridDim.x * LZ_THREADS) {
        const auto a = x[i], b = y[i];
        re += (double)a.x * (double)b.x + (double)a.y * (double)b.y;
        im += (double)a.x * (double)b.y - (double)a.y * (double)b.x;
    }
    block_sum2<T>(re, im);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = re; partial[2 * blockIdx.x + 1] = im; }
}

// One CTA: dst[0] = Re(sum of partials) (take_sqrt == 0) or sqrt of it (take_sqrt == 1).
__global__ void __launch_bounds__(32) lz_finalize_kernel(const double* __restrict__ partial, int n, double* dst, int take_sqrt)
{
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int b = 0; b < n; ++b) s += partial[2 * b];
        dst[0] = take_sqrt ? sqrt(s) : s;
    }
}

// w = w - alpha v - beta_prev v_prev, and the partial squared norm of the new w.
template <typename T>
__global__ void __launch_bounds__(LZ_THREADS) lz_update_kernel(int64_t D, typename Cplx<T>::type* __restrict__ w,
                                                               const typename Cplx<T>::type* __restrict__ v,
                                                               const typename Cplx<T>::type* __restrict__ v_prev,
                                                               const double* __restrict__ alpha, const double* __restrict__ beta_prev,
                                                               double* __restrict__ partial)
{
    using CT = typename Cplx<T>::type;
    const double a = alpha[0], bp = beta_prev ? beta_prev[0] : 0.0;
    double re = 0.0, im = 0.0;
    for (int64_t i = blockIdx.x * (int64_t)LZ_THREADS + threadIdx.x; i < D; i += (int64_t)gridDim.x * LZ_THREADS) {
        const CT wv = w[i], vv = v[i];
        double xr = (double)wv.x - a * (double)vv.x, xi = (double)wv.y - a * (double)vv.y;
        if (beta_prev) {
            const CT pv = v_prev[i];
            xr -= bp * (double)pv.x;
            xi -= bp * (double)pv.y;
        }
        CT o;
        o.x = (T)xr;
        o.y = (T)xi;
        w[i] = o;
        re += (double)o.x * (double)o.x + (double)o.y * (double)o.y;
    }
    block_sum2<T>(re, im);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = re; partial[2 * blockIdx.x + 1] = 0.0; }
}

// dst = src / scale[0]
template <typename T>
__global__ void __launch_bounds__(LZ_THREADS) lz_scale_kernel(int64_t D, const typename Cplx<T>::type* __restrict__ src,
                                                              typename Cplx<T>::type* __restrict__ dst, const double* __restrict__ scale)
{
    using CT = typename Cplx<T>::type;
    const double inv = 1.0 / scale[0];
    for (int64_t i = blockIdx.x * (int64_t)LZ_THREADS + threadIdx.x; i < D; i += (int64_t)gridDim.x * LZ_THREADS) {
        const CT s = src[i];
        CT o;
        o.x = (T)((double)s.x * inv);
        o.y = (T)((double)s.y * inv);
        dst[i] = o;
    }
}

template <typename T> static int lz_dot_t(mfh_handle h, const void* x, const void* y, double* partial, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    lz_dot_kernel<T><<<LZ_BLOCKS, LZ_THREADS, 0, st>>>(h->D, (const CT*)x, (const CT*)y, partial);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}
int launch_lz_dot(mfh_handle h, const void* x, const void* y, double* partial, double* dst, int take_sqrt, cudaStream_t st)
{
    int rc = h->dtype == MFH_C128 ? lz_dot_t<double>(h, x, y, partial, st) : lz_dot_t<float>(h, x, y, partial, st);
    if (rc) return rc;
    lz_finalize_kernel<<<1, 32, 0, st>>>(partial, LZ_BLOCKS, dst, take_sqrt);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}
int launch_lz_update(mfh_handle h, void* w, const void* v, const void* v_prev, const double* alpha, const double* beta_prev,
                     double* partial, double* beta_dst, cudaStream_t st)
{
    if (h->dtype == MFH_C128)
        lz_update_kernel<double><<<LZ_BLOCKS, LZ_THREADS, 0, st>>>(h->D, (double2*)w, (const double2*)v, (const double2*)v_prev,
                                                                   alpha, beta_prev, partial);
    else
        lz_update_kernel<float><<<LZ_BLOCKS, LZ_THREADS, 0, st>>>(h->D, (float2*)w, (const float2*)v, (const float2*)v_prev,
                                                                  alpha, beta_prev, partial);
    MFH_CUDA_CHECK(cudaGetLastError());
    lz_finalize_kernel<<<1, 32, 0, st>>>(partial, LZ_BLOCKS, beta_dst, 1);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}
int launch_lz_scale(mfh_handle h, const void* src, void* dst, const double* scale, cudaStream_t st)
{
    if (h->dtype == MFH_C128)
        lz_scale_kernel<double><<<LZ_BLOCKS, LZ_THREADS, 0, st>>>(h->D, (const double2*)src, (double2*)dst, scale);
    else
        lz_scale_kernel<float><<<LZ_BLOCKS, LZ_THREADS, 0, st>>>(h->D, (const float2*)src, (float2*)dst, scale);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}
int lz_partial_doubles() { return 2 * LZ_BLOCKS; }

}  // namespace mfh

// mfh_cached.cu -- cached-block streaming matvec: phi^[n] += sum_{m cached} C^[n,m] psi^[m]
// reading HBM-resident blocks (P:177-183 full / partial cache).
//
// HBM-bound: 16 B (c128) / 8 B (c64) of matrix per 4 FMAs.  Cache layout: block-major, each block
// row-major B x B interleaved complex, so a row of a block is one contiguous run of B entries.
// A CTA owns ROWS whole rows of the operator (no atomics, no cross-CTA sums): warp w streams its
// rows with 128-bit non-allocating loads, several independent loads in flight per lane; psi^[m]
// is staged once per CTA per column block in shared memory and shared by all warps.
#include <algorithm>
#include "mfh_internal.cuh"

namespace mfh {

__device__ __forceinline__ double2 ldg_stream(const double2* p)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float4 ldg_stream(const float4* p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p));
    return v;
}

template <typename T> struct CachedParams {
    int32_t B, n_blk, slot_cache;
    int64_t D;
    const int32_t* cache_slot;
    const typename Cplx<T>::type* cache;
    const typename Cplx<T>::type* psi;
    typename Cplx<T>::type* work;
};

constexpr int CACHED_WARPS = 8;
constexpr int CACHED_RPW = 2;                         // rows per warp
constexpr int CACHED_ROWS = CACHED_WARPS * CACHED_RPW;
constexpr int CACHED_U = 4;                           // independent loads per row per lane

// ---- complex128: one 16-byte load = one entry ----
__global__ void __launch_bounds__(32 * CACHED_WARPS) cached_kernel_c128(const CachedParams<double> P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* psis = reinterpret_cast<double2*>(smem_raw);   // [B]
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int B = P.B;
    const int64_t row0 = (int64_t)blockIdx.x * CACHED_ROWS;
    const int n = (int)(row0 / B);
    const int a0 = (int)(row0 % B) + w * CACHED_RPW;
    double accr[CACHED_RPW], acci[CACHED_RPW];
#pragma unroll
    for (int r = 0; r < CACHED_RPW; ++r) accr[r] = acci[r] = 0.0;

    for (int m = 0; m < P.n_blk; ++m) {
        const int32_t slot = P.cache_slot[n * P.n_blk + m];
        if (slot < 0) continue;
        __syncthreads();
        for (int c = tid; c < B; c += 32 * CACHED_WARPS) psis[c] = P.psi[(size_t)m * B + c];
        __syncthreads();
        const double2* rowp = P.cache + (size_t)slot * B * B + (size_t)a0 * B;
        for (int c = lane; c < B; c += 32 * CACHED_U) {
            double2 hv[CACHED_RPW][CACHED_U];
#pragma unroll
            for (int r = 0; r < CACHED_RPW; ++r)
#pragma unroll
                for (int u = 0; u < CACHED_U; ++u)
                    if (c + 32 * u < B) hv[r][u] = ldg_stream(rowp + (size_t)r * B + c + 32 * u);
#pragma unroll
            for (int u = 0; u < CACHED_U; ++u) {
                if (c + 32 * u < B) {
                    const double2 p = psis[c + 32 * u];
#pragma unroll
                    for (int r = 0; r < CACHED_RPW; ++r) {
                        accr[r] = fma(hv[r][u].x, p.x, accr[r]);
                        accr[r] = fma(-hv[r][u].y, p.y, accr[r]);
                        acci[r] = fma(hv[r][u].x, p.y, acci[r]);
                        acci[r] = fma(hv[r][u].y, p.x, acci[r]);
                    }
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < CACHED_RPW; ++r) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            accr[r] += __shfl_xor_sync(0xffffffffu, accr[r], o);
            acci[r] += __shfl_xor_sync(0xffffffffu, acci[r], o);
        }
        if (lane == 0)
            P.work[(size_t)P.slot_cache * P.D + row0 + w * CACHED_RPW + r] = double2{accr[r], acci[r]};
    }
}

// ---- complex64: one 16-byte load = two entries ----
__global__ void __launch_bounds__(32 * CACHED_WARPS) cached_kernel_c64(const CachedParams<float> P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* psis = reinterpret_cast<float4*>(smem_raw);   // [B/2] pairs of entries
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int B = P.B, B2 = P.B / 2;
    const int64_t row0 = (int64_t)blockIdx.x * CACHED_ROWS;
    const int n = (int)(row0 / B);
    const int a0 = (int)(row0 % B) + w * CACHED_RPW;
    float accr[CACHED_RPW], acci[CACHED_RPW];
#pragma unroll
    for (int r = 0; r < CACHED_RPW; ++r) accr[r] = acci[r] = 0.0f;

    for (int m = 0; m < P.n_blk; ++m) {
        const int32_t slot = P.cache_slot[n * P.n_blk + m];
        if (slot < 0) continue;
        __syncthreads();
        const float4* psrc = reinterpret_cast<const float4*>(P.psi + (size_t)m * B);
        for (int c = tid; c < B2; c += 32 * CACHED_WARPS) psis[c] = psrc[c];
        __syncthreads();
        const float4* rowp = reinterpret_cast<const float4*>(P.cache + (size_t)slot * B * B + (size_t)a0 * B);
        for (int c = lane; c < B2; c += 32 * CACHED_U) {
            float4 hv[CACHED_RPW][CACHED_U];
#pragma unroll
            for (int r = 0; r < CACHED_RPW; ++r)
#pragma unroll
                for (int u = 0; u < CACHED_U; ++u)
                    if (c + 32 * u < B2) hv[r][u] = ldg_stream(rowp + (size_t)r * B2 + c + 32 * u);
#pragma unroll
            for (int u = 0; u < CACHED_U; ++u) {
                if (c + 32 * u < B2) {
                    const float4 p = psis[c + 32 * u];
#pragma unroll
                    for (int r = 0; r < CACHED_RPW; ++r) {
                        const float4 hh = hv[r][u];
                        accr[r] = fmaf(hh.x, p.x, accr[r]);
                        accr[r] = fmaf(-hh.y, p.y, accr[r]);
                        acci[r] = fmaf(hh.x, p.y, acci[r]);
                        acci[r] = fmaf(hh.y, p.x, acci[r]);
                        accr[r] = fmaf(hh.z, p.z, accr[r]);
                        accr[r] = fmaf(-hh.w, p.w, accr[r]);
                        acci[r] = fmaf(hh.z, p.w, acci[r]);
                        acci[r] = fmaf(hh.w, p.z, acci[r]);
                    }
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < CACHED_RPW; ++r) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            accr[r] += __shfl_xor_sync(0xffffffffu, accr[r], o);
            acci[r] += __shfl_xor_sync(0xffffffffu, acci[r], o);
        }
        if (lane == 0)
            P.work[(size_t)P.slot_cache * P.D + row0 + w * CACHED_RPW + r] = float2{accr[r], acci[r]};
    }
}

int launch_cached(mfh_handle h, const void* psi, cudaStream_t st)
{
    const Plan& p = h->plan;
    if (p.n_cached == 0) return MFH_OK;
    if (p.k != 1) {
        set_error("cached blocks with k > 1 are not supported yet");
        return MFH_ERR_UNSUPPORTED;
    }
    const unsigned grid = (unsigned)(h->D / CACHED_ROWS);
    static bool attr_done = false;
    if (!attr_done) {
        MFH_CUDA_CHECK(cudaFuncSetAttribute(cached_kernel_c128, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            MFH_MAX_B * 16));
        MFH_CUDA_CHECK(cudaFuncSetAttribute(cached_kernel_c64, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            MFH_MAX_B * 8));
        attr_done = true;
    }
    if (h->dtype == MFH_C128) {
        CachedParams<double> P{p.B, p.n_blk, p.slot_cache, h->D, h->d_cache_slot,
                               (const double2*)h->d_cache, (const double2*)psi, (double2*)h->d_work};
        cached_kernel_c128<<<grid, 32 * CACHED_WARPS, (size_t)p.B * 16, st>>>(P);
    } else {
        CachedParams<float> P{p.B, p.n_blk, p.slot_cache, h->D, h->d_cache_slot,
                              (const float2*)h->d_cache, (const float2*)psi, (float2*)h->d_work};
        cached_kernel_c64<<<grid, 32 * CACHED_WARPS, (size_t)p.B * 8, st>>>(P);
    }
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

}  // namespace mfh

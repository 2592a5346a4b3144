// mfh_proc.cu -- generator-side kernels: Philox debug export, block materialisation / cache fill,
// H0 diagonal, and the fused generate-and-apply kernels (single vector with Hermitian reuse,
// k vectors one-sided).  PAPER.md Eq. 7, Eq. 8, Eq. 11.
#include <algorithm>
#include "mfh_internal.cuh"

namespace mfh {

template <typename T> static Scales<T> make_scales(int64_t D)
{
    Scales<T> s;
    s.off = (T)(1.0 / sqrt(2.0 * (double)D));
    s.diag = (T)(1.0 / sqrt((double)D));
    return s;
}

// --------------------------------------------------------------------------------------------
// Debug: raw words for (i,j) pairs.
// --------------------------------------------------------------------------------------------
__global__ void philox_debug_kernel(PhiloxKeys K, uint32_t stream_id, const uint32_t* __restrict__ i,
                                    const uint32_t* __restrict__ j, int64_t n,
                                    uint32_t* __restrict__ words)
{
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n;
         t += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t a = i[t], b = j[t];
        uint32_t x0, x1, x2, x3;
        philox4x32_10(K, min(a, b), max(a, b), stream_id, 0u, x0, x1, x2, x3);
        reinterpret_cast<uint4*>(words)[t] = make_uint4(x0, x1, x2, x3);
    }
}

int launch_philox_debug(uint64_t seed, uint32_t stream_id, const uint32_t* i, const uint32_t* j,
                        int64_t n, uint32_t* words, cudaStream_t st)
{
    if (n <= 0) return MFH_OK;
    const int threads = 256;
    const int blocks = (int)std::min<int64_t>((n + threads - 1) / threads, 148 * 8);
    philox_debug_kernel<<<blocks, threads, 0, st>>>(make_philox_keys(seed), stream_id, i, j, n, words);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// --------------------------------------------------------------------------------------------
// Block materialisation (test export) and cache fill: one dense B x B block per blockIdx.x,
// rows strided over blockIdx.y, columns over the threads (coalesced 16-byte stores).
// --------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) fill_kernel(PhiloxKeys K, Scales<T> S, int32_t B, int32_t n_blk,
                                                   const int32_t* __restrict__ cache_slot,
                                                   int32_t single_n, int32_t single_m,
                                                   typename Cplx<T>::type* __restrict__ out)
{
    using CT = typename Cplx<T>::type;
    int32_t n, m;
    size_t base;
    if (cache_slot) {
        const int32_t slot = cache_slot[blockIdx.x];
        if (slot < 0) return;
        n = blockIdx.x / n_blk;
        m = blockIdx.x % n_blk;
        base = (size_t)slot * B * B;
    } else {
        n = single_n;
        m = single_m;
        base = 0;
    }
    for (int32_t a = blockIdx.y; a < B; a += gridDim.y) {
        const uint32_t i = (uint32_t)n * B + a;
        CT* row = out + base + (size_t)a * B;
        for (int32_t b = threadIdx.x; b < B; b += blockDim.x) {
            T hr, hi;
            entry_any<T>(K, S, i, (uint32_t)m * B + b, hr, hi);
            CT v;
            v.x = hr;
            v.y = hi;
            row[b] = v;
        }
    }
}

int launch_fill_block(mfh_handle h, int32_t B, int32_t n, int32_t m, void* out, cudaStream_t st)
{
    const PhiloxKeys K = make_philox_keys(h->seed);
    dim3 grid(1, std::min(B, 1024));
    if (h->dtype == MFH_C128)
        fill_kernel<double><<<grid, 256, 0, st>>>(K, make_scales<double>(h->D), B, 0, nullptr, n, m,
                                                   (double2*)out);
    else
        fill_kernel<float><<<grid, 256, 0, st>>>(K, make_scales<float>(h->D), B, 0, nullptr, n, m,
                                                  (float2*)out);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_fill_cache(mfh_handle h, cudaStream_t st)
{
    const Plan& p = h->plan;
    if (p.n_cached == 0) return MFH_OK;
    const PhiloxKeys K = make_philox_keys(h->seed);
    dim3 grid(p.n_blk * p.n_blk, std::min(p.B, 64));
    if (h->dtype == MFH_C128)
        fill_kernel<double><<<grid, 256, 0, st>>>(K, make_scales<double>(h->D), p.B, p.n_blk,
                                                   h->d_cache_slot, 0, 0, (double2*)h->d_cache);
    else
        fill_kernel<float><<<grid, 256, 0, st>>>(K, make_scales<float>(h->D), p.B, p.n_blk,
                                                  h->d_cache_slot, 0, 0, (float2*)h->d_cache);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// --------------------------------------------------------------------------------------------
// H0 diagonal of configs[2]: h0_i = 2u - 1, u = (x0 + 1/2) 2^-32, ctr = (i, i, stream 1, 0).
// --------------------------------------------------------------------------------------------
template <typename T>
__global__ void h0_kernel(PhiloxKeys K, int64_t D, T* __restrict__ h0)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < D;
         i += (int64_t)gridDim.x * blockDim.x) {
        uint32_t x0, x1, x2, x3;
        philox4x32_10(K, (uint32_t)i, (uint32_t)i, 1u, 0u, x0, x1, x2, x3);
        const double d0 = __hiloint2double(0x43300000, (int)x0);
        const double u = fma(d0, 0x1p-32, -(0x1p52 - 0.5) * 0x1p-32);
        h0[i] = (T)(2.0 * u - 1.0);
    }
}

int launch_h0(mfh_handle h, void* out, cudaStream_t st)
{
    const PhiloxKeys K = make_philox_keys(h->seed_h0);
    const int blocks = (int)std::min<int64_t>((h->D + 255) / 256, 148 * 8);
    if (h->dtype == MFH_C128)
        h0_kernel<double><<<blocks, 256, 0, st>>>(K, h->D, (double*)out);
    else
        h0_kernel<float><<<blocks, 256, 0, st>>>(K, h->D, (float*)out);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

// --------------------------------------------------------------------------------------------
// Fused generate-and-apply, ONE vector, Hermitian reuse (Eq. 11).
//
// Work item = rows [row0, row0+nrows) of block n  x  all columns of block m  (n <= m, or any
// (n,m) for a one-sided item).  A CTA of W warps walks macro tiles of 32W x 32W entries; inside
// a macro tile warp w owns the 32 rows w*32.. and at step t works on column sub-tile (w+t)%W, so
// in every step each warp has its own rows AND its own columns.  Inside a 32x32 sub-tile lane l
// owns row l and at step s handles column (l+s)%32: the entry H_ij (i<j) is generated once in
// registers and used twice,
//     row side     phi_i += H_ij psi_j              (accumulator stays in lane l)
//     column side  phi_j += conj(H_ij) psi_i        (accumulator rotates lane l+1 -> l each step)
// so after 32 steps lane l holds the complete column-l sum of the sub-tile: no atomics anywhere.
// Column sums are added to a shared-memory array (exclusive per step, barrier between steps),
// row sums live in registers across the whole item.  Results go to partial slots that the
// reduce kernel adds in a fixed order (deterministic).
// --------------------------------------------------------------------------------------------
template <typename T> struct ProcParams {
    PhiloxKeys K;
    Scales<T> S;
    int32_t B, n_blk, n_items, slot_row0;
    int64_t D;
    const ProcItem* items;
    const typename Cplx<T>::type* psi;
    typename Cplx<T>::type* work;   // [n_slots][D]
    int32_t* counter;
};

template <typename T, int W>
__global__ void __launch_bounds__(32 * W) proc_single_kernel(const ProcParams<T> P)
{
    using CT = typename Cplx<T>::type;
    constexpr int MT = 32 * W;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CT* colsum = reinterpret_cast<CT*>(smem_raw);   // [B]  column-side sums of the item
    CT* psic = colsum + P.B;                        // [MT] psi of the current column macro tile
    __shared__ int s_item;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int B = P.B;

    for (;;) {
        if (tid == 0) s_item = atomicAdd(P.counter, 1);
        __syncthreads();
        const int it = s_item;
        __syncthreads();
        if (it >= P.n_items) break;
        const ProcItem I = P.items[it];
        const bool one_sided_item = (I.kind == PAIR_ONE_SIDED);
        const bool diag_item = (I.kind == PAIR_DIAG);
        for (int c = tid; c < B; c += MT) colsum[c] = CT{T(0), T(0)};
        const int ncm = B / MT;

        for (int rloc = I.row0; rloc < I.row0 + I.nrows; rloc += MT) {
            const uint32_t i = (uint32_t)I.n * B + rloc + w * 32 + lane;
            const CT psi_i = P.psi[i];
            T accr = T(0), acci = T(0);
            const int rmac = rloc / MT;
            for (int cm = diag_item ? rmac : 0; cm < ncm; ++cm) {
                __syncthreads();
                psic[tid] = P.psi[(size_t)I.m * B + cm * MT + tid];
                __syncthreads();
                const bool mdiag = diag_item && (cm == rmac);
#pragma unroll 1
                for (int t = 0; t < W; ++t) {
                    const int cs = (w + t) & (W - 1);
                    const uint32_t j0 = (uint32_t)I.m * B + cm * MT + cs * 32;
                    const CT* pc = psic + cs * 32;
                    if (one_sided_item || (mdiag && cs == w)) {
#pragma unroll 2
                        for (int s = 0; s < 32; ++s) {
                            T hr, hi;
                            entry_any<T>(P.K, P.S, i, j0 + s, hr, hi);
                            const CT p = pc[s];
                            accr = fma(hr, p.x, accr);
                            accr = fma(-hi, p.y, accr);
                            acci = fma(hr, p.y, acci);
                            acci = fma(hi, p.x, acci);
                        }
                    } else if (!(mdiag && cs < w)) {
                        T cr = T(0), ci = T(0);
#pragma unroll 2
                        for (int s = 0; s < 32; ++s) {
                            const int c = (lane + s) & 31;
                            T hr, hi;
                            entry_upper<T>(P.K, P.S, i, j0 + c, hr, hi);
                            const CT p = pc[c];
                            accr = fma(hr, p.x, accr);
                            accr = fma(-hi, p.y, accr);
                            acci = fma(hr, p.y, acci);
                            acci = fma(hi, p.x, acci);
                            cr = fma(hr, psi_i.x, cr);     // conj(H_ij) psi_i
                            cr = fma(hi, psi_i.y, cr);
                            ci = fma(hr, psi_i.y, ci);
                            ci = fma(-hi, psi_i.x, ci);
                            cr = __shfl_sync(0xffffffffu, cr, (lane + 1) & 31);
                            ci = __shfl_sync(0xffffffffu, ci, (lane + 1) & 31);
                        }
                        CT& dst = colsum[cm * MT + cs * 32 + lane];
                        dst.x += cr;
                        dst.y += ci;
                    }
                    __syncthreads();
                }
            }
            P.work[(size_t)(P.slot_row0 + I.m) * P.D + i] = CT{accr, acci};
        }
        __syncthreads();
        if (I.col_slot >= 0) {
            CT* dst = P.work + (size_t)I.col_slot * P.D + (size_t)I.m * B;
            for (int c = tid; c < B; c += MT) dst[c] = colsum[c];
        }
    }
}

template <typename T, int W>
static int launch_proc_single_t(mfh_handle h, const void* psi, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    const Plan& p = h->plan;
    ProcParams<T> P;
    P.K = make_philox_keys(h->seed);
    P.S = make_scales<T>(h->D);
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.n_items = (int32_t)p.items.size();
    P.slot_row0 = p.slot_row0;
    P.D = h->D;
    P.items = h->d_items;
    P.psi = (const CT*)psi;
    P.work = (CT*)h->d_work;
    P.counter = h->d_counter;
    const size_t smem = (size_t)(p.B + 32 * W) * sizeof(CT);
    auto kern = proc_single_kernel<T, W>;
    static bool attr_done = false;
    if (!attr_done) {
        MFH_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)((MFH_MAX_B + 32 * W) * sizeof(CT))));
        attr_done = true;
    }
    int per_sm = 1;
    MFH_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 32 * W, smem));
    if (per_sm < 1) per_sm = 1;
    const int grid = std::min<int>(P.n_items, h->sm_count * per_sm);
    MFH_CUDA_CHECK(cudaMemsetAsync(h->d_counter, 0, sizeof(int32_t), st));
    kern<<<grid, 32 * W, smem, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_proc_single(mfh_handle h, const void* psi, cudaStream_t st)
{
    if (h->plan.items.empty()) return MFH_OK;
    const bool f64 = (h->dtype == MFH_C128);
    switch (h->plan.warps) {
    case 8: return f64 ? launch_proc_single_t<double, 8>(h, psi, st) : launch_proc_single_t<float, 8>(h, psi, st);
    case 4: return f64 ? launch_proc_single_t<double, 4>(h, psi, st) : launch_proc_single_t<float, 4>(h, psi, st);
    case 2: return f64 ? launch_proc_single_t<double, 2>(h, psi, st) : launch_proc_single_t<float, 2>(h, psi, st);
    case 1: return f64 ? launch_proc_single_t<double, 1>(h, psi, st) : launch_proc_single_t<float, 1>(h, psi, st);
    }
    set_error("unsupported warps per CTA %d", h->plan.warps);
    return MFH_ERR_INVALID_ARG;
}

// --------------------------------------------------------------------------------------------
// Fused generate-and-apply, k vectors (coupling scans, Eq. 12): every V entry is
// generated ONCE per apply and multiplied into all k columns.  One-sided: lane = row, the CTA
// owns 32W rows over all uncached column blocks, the psi rows of a column chunk are staged in
// shared memory and read as broadcasts; k accumulators per lane stay in registers, so the
// result is written once with no partial sums over m.
// --------------------------------------------------------------------------------------------
template <typename T> struct MultiParams {
    PhiloxKeys K;
    Scales<T> S;
    int32_t B, n_blk, k, slot_multi;
    int64_t D;
    const int32_t* cache_slot;
    const typename Cplx<T>::type* psi;   // [D][k]
    typename Cplx<T>::type* work;        // [n_slots][D][k]
};

template <typename T, int KT, int W>
__global__ void __launch_bounds__(32 * W) proc_multi_kernel(const MultiParams<T> P)
{
    using CT = typename Cplx<T>::type;
    constexpr int CH = 32;                         // columns per staged chunk
    __shared__ __align__(16) CT psis[CH][KT];
    const int tid = threadIdx.x;
    const uint32_t i = blockIdx.x * (32 * W) + tid;
    const int n = (int)(i / (uint32_t)P.B);
    const int k = P.k;
    CT acc[KT];
#pragma unroll
    for (int v = 0; v < KT; ++v) acc[v] = CT{T(0), T(0)};

    for (int m = 0; m < P.n_blk; ++m) {
        if (P.cache_slot[n * P.n_blk + m] >= 0) continue;   // cached blocks: streaming kernel
        for (int c0 = 0; c0 < P.B; c0 += CH) {
            const uint32_t j0 = (uint32_t)m * P.B + c0;
            __syncthreads();
            for (int e = tid; e < CH * KT; e += 32 * W) {
                const int c = e / KT, v = e % KT;
                psis[c][v] = (v < k) ? P.psi[(size_t)(j0 + c) * k + v] : CT{T(0), T(0)};
            }
            __syncthreads();
#pragma unroll 2
            for (int c = 0; c < CH; ++c) {
                T hr, hi;
                entry_any<T>(P.K, P.S, i, j0 + c, hr, hi);
#pragma unroll
                for (int v = 0; v < KT; ++v) {
                    const CT p = psis[c][v];
                    acc[v].x = fma(hr, p.x, acc[v].x);
                    acc[v].x = fma(-hi, p.y, acc[v].x);
                    acc[v].y = fma(hr, p.y, acc[v].y);
                    acc[v].y = fma(hi, p.x, acc[v].y);
                }
            }
        }
    }
    CT* dst = P.work + ((size_t)P.slot_multi * P.D + i) * k;
#pragma unroll
    for (int v = 0; v < KT; ++v)
        if (v < k) dst[v] = acc[v];
}

template <typename T, int KT>
static int launch_proc_multi_t(mfh_handle h, const void* psi, cudaStream_t st)
{
    using CT = typename Cplx<T>::type;
    const Plan& p = h->plan;
    MultiParams<T> P;
    P.K = make_philox_keys(h->seed);
    P.S = make_scales<T>(h->D);
    P.B = p.B;
    P.n_blk = p.n_blk;
    P.k = p.k;
    P.slot_multi = p.slot_multi;
    P.D = h->D;
    P.cache_slot = h->d_cache_slot;
    P.psi = (const CT*)psi;
    P.work = (CT*)h->d_work;
    // 32W rows per CTA must divide B; prefer 128-row CTAs, fall back to one warp.
    if (p.B % 128 == 0)
        proc_multi_kernel<T, KT, 4><<<(unsigned)(h->D / 128), 128, 0, st>>>(P);
    else
        proc_multi_kernel<T, KT, 1><<<(unsigned)(h->D / 32), 32, 0, st>>>(P);
    MFH_CUDA_CHECK(cudaGetLastError());
    return MFH_OK;
}

int launch_proc_multi(mfh_handle h, const void* psi, cudaStream_t st)
{
    const int k = h->plan.k;
    const bool f64 = (h->dtype == MFH_C128);
    if (k <= 2) return f64 ? launch_proc_multi_t<double, 2>(h, psi, st) : launch_proc_multi_t<float, 2>(h, psi, st);
    if (k <= 4) return f64 ? launch_proc_multi_t<double, 4>(h, psi, st) : launch_proc_multi_t<float, 4>(h, psi, st);
    if (k <= 8) return f64 ? launch_proc_multi_t<double, 8>(h, psi, st) : launch_proc_multi_t<float, 8>(h, psi, st);
    return f64 ? launch_proc_multi_t<double, 16>(h, psi, st) : launch_proc_multi_t<float, 16>(h, psi, st);
}

}  // namespace mfh
